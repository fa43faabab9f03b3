/*
 * octo_fmm.h -- C ABI of the B200-native FMM cell-to-cell interaction step.
 *
 * The operation (PAPER.md = arxiv 2101.08226, section 2.2 "Gravity Update and the Angular
 * Momentum Correction", L123-139): on a uniform level of cells grouped in 8x8x8 sub-grids
 * (L287), every cell A accumulates an order-3 local Taylor expansion of the potential
 * (20 FP64 coefficients) from the order-3 multipole moments (20 FP64 components) of every
 * same-level cell B that is well separated from A while their parents are not (opening
 * criterion, Eq. 15), plus the angular-momentum-conserving correction (L127) and
 * the monopole (leaf) variant.  Domain is isolated (L321), G = 1 (L363).  The formulas the
 * paper defers to Dehnen (2000) / Marcello et al. (2016) are restated in DESIGN.md.
 *
 * Conventions
 *   - cell index (i,j,k), x fastest; geometric centre x = origin + (i + 1/2) h.
 *   - moments: raw Cartesian moments about the cell's expansion centre z = x + delta,
 *       M^(n) = sum_p m_p (y_p - z)^{(x)n}, n = 0..3, 20 unique components in the order
 *       [0] [x y z] [xx xy xz yy yz zz] [xxx xxy xxz xyy xyz xzz yyy yyz yzz zzz],
 *       no factorials or multiplicities folded in;  layout [20][nz][ny][nx] (SoA).
 *   - com_off: delta = z - x_cell, layout [3][nz][ny][nx]; |delta_c| <= h/2.
 *   - expansions: L^(n) = d^n phi / dx^n at z_A, same 20-slot order, layout
 *       [20][oz][oy][ox] over the output region; with am_correction the correction is folded
 *       into L^(1); Lcorr [3][oz][oy][ox] returns it alone.
 *   - monopole kind: moments = mass [1][nz][ny][nx] at the geometric centres, output
 *       [4][oz][oy][ox] = (phi, g_x, g_y, g_z),  phi = -sum m/|R|,  g = -sum m R/|R|^3.
 *   - pair separation, in this operation order:
 *       R_c = (double)(i_A,c - i_B,c) * h + (delta_A,c - delta_B,c).
 *
 * Memory and ownership: every pointer marked "device" is device memory on cfg.device owned by
 * the caller; the library never allocates or frees device memory (the caller lends it a
 * workspace) and never synchronises the stream except in octo_fmm_destroy, octo_fmm_status, the
 * counters that read a device word, the *_host entry points and (MONOPOLE handles, tree) create.  All work is enqueued on cfg.stream (a cudaStream_t).  Inputs may be reused
 * by the caller once the stream has passed set_moments; outputs are complete once the stream
 * has passed get_expansions.  One handle is not thread-safe; DIFFERENT handles may be driven from
 * different streams and host threads at the same time.  Everything that depends on a handle's cell
 * width travels with its launches; the interaction lists (a function of theta and kind only) are
 * kept in one constant-memory bank per device, and the library orders an upload of other lists
 * against the kernels of other streams that still read the previous ones (events, no host
 * synchronisation): handles with the same theta and kind share the bank and run concurrently,
 * handles with different lists are serialised on the device.
 *
 * Errors: every call returns an OCTO_FMM_* status; nothing throws or aborts.
 * There is no CPU fallback: without a usable CUDA device create() fails with OCTO_FMM_ECUDA.
 */
#ifndef OCTO_FMM_H
#define OCTO_FMM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct octo_fmm octo_fmm_t; /* opaque handle */

enum { OCTO_FMM_OK = 0, OCTO_FMM_EINVAL = 1, OCTO_FMM_ESTATE = 2, OCTO_FMM_ENOMEM = 3, OCTO_FMM_ECUDA = 4,
       OCTO_FMM_EMASS = 5 /* am_correction with a target cell of mass <= 0 (division M_B/M_A, L127) */,
       OCTO_FMM_ESIZE = 6 /* octo_fmm_interact_static: the grid has more cells than OCTO_FMM_STATIC_MAX_CELLS */ };
enum { OCTO_FMM_MULTIPOLE = 0, OCTO_FMM_MONOPOLE = 1 };

typedef struct {
    int n[3];                  /* cells per axis (x,y,z), each a positive multiple of 8 (8^3 sub-grids, L287) */
    int out_lo[3], out_hi[3];  /* target region in cells, 8-aligned; lo = hi = 0 -> the whole grid           */
    double h;                  /* cell width                                                                  */
    double origin[3];          /* lower corner of the grid (kept for the caller; results do not depend on it) */
    double theta;              /* opening angle, 1/3 < theta < 1: halo reach <= 5 cells (theta_min, L137)     */
    int kind;                  /* OCTO_FMM_MULTIPOLE | OCTO_FMM_MONOPOLE                                      */
    int am_correction;         /* 0/1, ignored for MONOPOLE                                                   */
    int device;                /* CUDA device ordinal                                                         */
    void *stream;              /* cudaStream_t, borrowed                                                      */
    void *workspace;           /* device memory, 256-byte aligned, borrowed for the handle's lifetime         */
    size_t workspace_bytes;    /* >= octo_fmm_workspace_bytes(cfg)                                            */
} octo_fmm_config;

/* Bytes of device workspace a handle for this configuration needs (0 on invalid configuration). */
size_t octo_fmm_workspace_bytes(const octo_fmm_config *cfg);

/* Builds the 8 per-parity interaction lists from Eq. 15 (L131-135) on the host and the TMA
 * descriptors of the workspace; no device allocation.  MONOPOLE handles also upload the tables of
 * the tensor-core kernel (weights of the 11^3 offsets, operand fragments) into the workspace and
 * synchronise cfg.stream once for it (the tables come from pageable host memory).  EINVAL: bad sizes
 * / theta / NULL / workspace too small or misaligned.  ECUDA: no usable device. */
int octo_fmm_create(const octo_fmm_config *cfg, octo_fmm_t **out);

/* Stage the sources: re-lays the caller's moments into the workspace
 * (asynchronously, on the stream).  moments: device, [20][nz][ny][nx] (MONOPOLE: [1][nz][ny][nx]);
 * com_off: device, [3][nz][ny][nx] (NULL for MONOPOLE, or for offset 0). */
int octo_fmm_set_moments(octo_fmm_t *h, const double *moments, const double *com_off);

/* The interaction step (a3-a5), asynchronous on the stream.  ESTATE before set_moments. */
int octo_fmm_interact(octo_fmm_t *h);

/* Copy the results out (a6), asynchronous on the stream.  L: device, [20] (MONOPOLE: [4]) x
 * out cells; Lcorr: device, [3] x out cells, or NULL.  ESTATE before interact. */
int octo_fmm_get_expansions(octo_fmm_t *h, double *L, double *Lcorr);

/* Optional: make interact() write its results straight into caller buffers (device, same shapes
 * as get_expansions; with Lcorr = NULL the correction alone stays in the workspace).  A later
 * get_expansions() with the same pointers then copies nothing.  L = NULL
 * restores the default (results kept in the workspace).  The buffers must stay valid until
 * the stream has passed the interact() calls that use them. */
int octo_fmm_bind_outputs(octo_fmm_t *h, double *L, double *Lcorr);

/* Synchronises the stream and releases the handle (not the workspace). */
int octo_fmm_destroy(octo_fmm_t *h);

/* ---- auxiliary ------------------------------------------------------------------------- */

/* Interaction list of parity class parity = px + 2 py + 4 pz, in (dz,dy,dx)-lexicographic order.
 * *count receives the list length; dxyz (may be NULL) must hold that many (dx,dy,dz) triples. */
int octo_fmm_get_stencil(const octo_fmm_t *h, int parity, int *count, signed char (*dxyz)[3]);

/* Host-only view (no device, no handle) of the operand tables of the tensor-core monopole kernels, for tests: the
 * table for opening angle theta, cell width h, list flavour leaf (0 = the list of Eq. 15, 1 = + the near field of
 * the complete solve) and which = 0..3 (the (y, z)-parity pair py + 2 pz of the four-output kernel: rows 0-3 =
 * (phi, gx, gy, gz) of the x-even target, rows 4-7 of its x-odd sibling) or 4 (potential-only kernel: row v = child
 * vx + 2 vy + 4 vz of one parent).  *nchunk chunks of 4 source positions; for chunk c, row i, slot k:
 * a[32 c + 4 i + k] = the weight (0 where the position is not in row i's list), off[32 c + 4 i + k] = the position's
 * offset in the mass tile, (sz * 26 + sy) * 28 + ((sx + 5) & 1) * 14 + ((sx + 5) >> 1) doubles, position (sx, sy, sz)
 * relative to the base target.  a, off: host, cap_chunks * 32 elements (NULL: only *nchunk). */
int octo_fmm_dmma_table(double theta, double h, int leaf, int which, int cap_chunks, int *nchunk, double *a, int *off);

/* Number of ordered in-domain (A,B) pairs one interact() evaluates (out-of-grid partners are
 * skipped: isolated boundary, L321). */
int octo_fmm_interaction_count(const octo_fmm_t *h, unsigned long long *n);

/* ---- f4: one uniform level sharded into z-slabs, the halo read from PEER MEMORY (the step needs
 * "boundary data from sibling sub-grids" -- here the sub-grids of the neighbouring ranks) ----
 * Rank r holds the z-layers of its slab in a handle of its own (n = {nx, ny, nz_local}; whole-slab output region).
 * octo_fmm_set_neighbours tells the handle where the staged source arrays of the slabs below (z < 0) and above
 * (z >= nz_local) live; octo_fmm_interact then treats the three slabs as one grid: the slab-fed kernel's TMA loads fetch
 * the layers within the stencil's reach straight from the neighbours' arrays -- over NVLink when those sit on another
 * GPU -- while it computes; there is no exchange step, no packing and no halo storage.  NULL = the isolated domain
 * boundary on that side (L321).  Results are identical to one handle over the three slabs (same kernel, same order).
 *   octo_fmm_peer: `sources`, `flags` = what octo_fmm_staged_sources returned for the neighbour's handle, as DEVICE
 *   pointers valid in the calling process (same process: as they are, with peer access enabled between the devices;
 *   another process: through the octo_fmm_ipc_* helpers below); nz = the neighbour's z-extent (>= 5).  The neighbour's
 *   handle must have the same nx, ny, h, theta, kind = MULTIPOLE and am_correction.  Pointers are borrowed.
 * Ordering is the caller's: every rank's set_moments must have COMPLETED (stream synchronised + a barrier across ranks)
 * before any rank's interact, and no rank may stage again before its neighbours' interact has completed.
 * Errors: EINVAL for a monopole handle, a handle whose output region is too small for the slab-fed kernel, nz < 5 or
 * null/misaligned pointers.  With neighbours set, octo_fmm_run_host and octo_fmm_interact_mixed return ESTATE.
 * octo_fmm_interaction_count counts the pairs with partners in the neighbouring slabs too. */
typedef struct octo_fmm_peer {
    const double *sources;
    const int *flags;
    int nz;
} octo_fmm_peer;
int octo_fmm_staged_sources(const octo_fmm_t *h, octo_fmm_peer *self);
int octo_fmm_set_neighbours(octo_fmm_t *h, const octo_fmm_peer *below, const octo_fmm_peer *above);

/* CUDA IPC plumbing for one process per GPU: export yields the 64-byte handle of the ALLOCATION that holds dev_ptr
 * (e.g. the workspace) and dev_ptr's offset in it; import maps that allocation into the calling process (peer access is
 * enabled lazily) and returns its base (for octo_fmm_ipc_close) and the pointer at the offset.  The exporter keeps the
 * memory alive until every importer has closed.  Host-side, synchronous; ECUDA if the memory cannot be shared (it must
 * come from cudaMalloc, which is what torch's caching allocator uses unless expandable segments are on). */
int octo_fmm_ipc_export(const void *dev_ptr, unsigned char handle[64], unsigned long long *offset);
int octo_fmm_ipc_import(const unsigned char handle[64], unsigned long long offset, void **base, void **dev_ptr);
int octo_fmm_ipc_close(void *base);

/* Synchronises the stream and reports device-side conditions of the last interact():
 * OCTO_FMM_EMASS if am_correction met a target mass <= 0, ECUDA on a CUDA error, else OK. */
int octo_fmm_status(octo_fmm_t *h);

/* Whole step with HOST buffers (pinned or pageable): H2D of moments/com_off into
 * scratch, set_moments, interact (writing into the scratch), D2H of L (and Lcorr if non-NULL), then
 * a stream synchronise.  For the multipole kind the step is pipelined over slabs of z-layers on two
 * internal copy streams, so that the copy in of slab c+1, the kernels of slab c and the copy out of
 * slab c-1 overlap (pinned host buffers are needed for the overlap, not for correctness); every
 * layer crosses the bus once per direction.  Returns OCTO_FMM_EMASS if the correction met a target
 * mass <= 0.  Afterwards the handle is in the "sources staged" state.
 * scratch: device, >= octo_fmm_host_scratch_bytes(cfg) bytes, borrowed for the call. */
size_t octo_fmm_host_scratch_bytes(const octo_fmm_config *cfg);
int octo_fmm_run_host(octo_fmm_t *h, const double *moments_host, const double *com_off_host,
                      double *L_host, double *Lcorr_host, void *scratch, size_t scratch_bytes);

/* The dipole terms.  Sources expanded about their centre of mass have M^(1) = 0 up to round-off, and the 27
 * terms that contain M^(1) then contribute nothing.  set_moments() checks on the device whether every cell
 * has |M^(1)_i| <= 4e-16 |M| h; if so interact() leaves those terms out (188 instead of 224 flop per
 * interaction), otherwise it evaluates them -- results agree with the general formula to round-off either
 * way.  octo_fmm_set_option(h, "dipole_terms", 1) forces the general path.  After set_moments(),
 * octo_fmm_dipole_terms_used() synchronises the stream and tells which path interact() takes. */
int octo_fmm_dipole_terms_used(octo_fmm_t *h, int *used);

/* One level of an ADAPTIVE mesh (a node "is either fully refined with eight child nodes
 * (an interior node) or not refined at all (a leaf node)"; the paper does not describe the gravity side of a
 * refinement boundary: DESIGN.md reading R8).  leaf: device, [nz][ny][nx] bytes, 1 = the cell belongs to a leaf
 * sub-grid (it has no children; hand it over as a point mass: M1 = M2 = M3 = 0, offset 0), 0 = to a refined one.
 * octo_fmm_interact_mixed() = octo_fmm_interact() (the list of Eq. 15, whatever the cells' kind) + the near-field
 * pairs nobody below this level will take: a cell B that is NOT well separated from A (and whose parent is not well
 * separated from A's) interacts with A here if A or B is a leaf.  Same pair formula, same outputs (get_expansions).
 * MULTIPOLE handles; asynchronous on the stream.  With octo_fmm_set_option(h, "mixed_count", 1) the call also counts
 * the ordered pairs it evaluates (they depend on leaf); octo_fmm_mixed_interaction_count() then synchronises the stream
 * and returns the number (ESTATE if the last octo_fmm_interact_mixed() did not count). */
int octo_fmm_interact_mixed(octo_fmm_t *h, const unsigned char *leaf);
int octo_fmm_mixed_interaction_count(octo_fmm_t *h, unsigned long long *n);

/* Options, for tests and profiling.  "kernel" = 0 staged (TMA + shared memory; default above 4096 target
 * cells), 1 direct (one cell per thread, global-memory loads; same pair arithmetic), 2 one warp per cell with
 * a warp-level reduction of the partial expansions (default up to 4096 target cells).
 * "dipole_terms" = 0 decided on the device (default), 1 always evaluated.
 * "mixed_count" = 1: octo_fmm_interact_mixed also counts its pairs (default 0).
 * "am_correction" = 0 / 1 (MULTIPOLE handles): switches the correction of cfg.am_correction for the following
 * set_moments() + interact() (the handle goes back to the "created" state) -- one handle and one workspace can
 * so serve a second right-hand side on the same centres (d(rho)/dt, L81-83: no correction) after the first.
 * "host_chunk" = output z-layers per pipeline slab of octo_fmm_run_host (default 12; 0 = one copy in, one
 * launch, one copy out).
 * "mono_kernel" (MONOPOLE handles) = 0 the sum as 8x8x4 FP64 tensor-core contractions (mma.sync m8n8k4.f64:
 * 16-cell row segments x 4 offsets per instruction; default), 1 the same sum with DFMAs.  Both follow the list
 * of Eq. 15 and agree to round-off (the summation order differs).  Unknown keys -> EINVAL. */
int octo_fmm_set_option(octo_fmm_t *h, const char *key, int value);

/* Launch facts of the interaction kernel the handle would run: grid, block, dynamic shared
 * memory bytes, registers per thread, number of kernels launched per interact(). */
int octo_fmm_launch_info(const octo_fmm_t *h, int *grid, int *block, int *smem_bytes, int *regs,
                         int *launches_per_interact);

/* FP64 ALU roofline probe: runs `iters` dependent-free DFMA chains on every SM of the device and
 * returns the measured FP64 FLOP/s (2 per DFMA), SM count and SM clock (kHz, device attribute).
 * scratch: device, >= 8 * 1024 * 1024 bytes. */
int octo_fmm_fp64_peak_probe(int device, void *stream, void *scratch, int iters, double *flops_per_s,
                             int *sm_count, int *clock_khz);

/* FP64 issue-rate probe with REGISTER operands, 12 warps per SM: mode 0 = DFMA with three fresh register
 * operands, 1 = DFMA repeating one operand in the same slot (operand-reuse cache), 2 = DMUL.  Returns
 * thread-level FP64 instructions per second (issue peak = SMs x 64 x clock).  It documents why the
 * interaction kernel's FP64 pipe is not 100 % busy.  scratch: device, >= 8 MiB. */
int octo_fmm_fp64_issue_probe(int device, void *stream, void *scratch, int mode, int iters, double *instr_per_s);

/* FP64 operations one multipole (kind 0) / monopole (kind 1) interaction executes in the kernel's inner loop, counted
 * in its SASS (DFMA = 2 flop, DADD/DMUL = 1, the reciprocal-square-root instruction not counted); see DESIGN.md
 * section 7.  These are the flops `bench.py` quotes its roofline on: 212 with the correction and the dipole terms since
 * round 2 (224 in round 1; the full-tensor definition needs about 400). */
int octo_fmm_flops_per_interaction(int kind, int am_correction, int *flops, int *fp64_instructions);
/* The same for a given path: dipole_terms = 0 is the path without the 27 dipole terms (multipole kind only). */
int octo_fmm_flops_per_interaction_path(int kind, int am_correction, int dipole_terms, int *flops, int *fp64_instructions);

const char *octo_fmm_version(void);

/* ---- the interaction step WITHOUT any allocation ------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it) and have no workspace to lend: the same step as octo_fmm_set_moments + octo_fmm_interact (PAPER.md L125-137,
 * multipole kind), one call, with its scratch (staged sources, flag words) in a static device array inside the library.
 * The library holds that array, OCTO_FMM_STATIC_MAX_CELLS x 344 bytes + 1.3 KB = 11.3 MB, on every GPU that loads it,
 * until the process exits.  The call allocates no device memory: no cudaMalloc / cudaFree / allocating library routine;
 * a call with a configuration other than the previous one's on that device builds a new handle in HOST memory and
 * first waits for the previous configuration's stream.
 *   cfg: as for octo_fmm_create (n multiples of 8, theta, h, am_correction, out_lo/out_hi, device, stream), kind =
 *   OCTO_FMM_MULTIPOLE; workspace and workspace_bytes are ignored.  moments [20][nz][ny][nx], com_off [3][nz][ny][nx]
 *   (NULL: geometric centres), L [20][out cells], Lcorr [3][out cells] or NULL: DEVICE pointers of the caller,
 *   borrowed for the call; the results are complete when cfg->stream has run the two kernels (the call does not wait).
 * Errors: OCTO_FMM_ESIZE if n[0] n[1] n[2] > OCTO_FMM_STATIC_MAX_CELLS (nothing is launched); EINVAL for a bad
 * configuration, the monopole kind or null moments / L; ECUDA.  octo_fmm_static_status(device) synchronises the stream
 * of the last call on that device and reports EMASS like octo_fmm_status (ESTATE before the first call).
 * EVERY call on a device shares the one array, which keeps the contents of the call before (the call clears what must
 * start at zero): calls serialise on the host, but two calls whose kernels OVERLAP on the GPU -- different streams
 * without an ordering between them -- race on it.  One stream, or an event between the calls. */
#define OCTO_FMM_STATIC_MAX_CELLS 32768 /* e.g. 32 x 32 x 32 */
int octo_fmm_static_max_cells(void);
int octo_fmm_interact_static(const octo_fmm_config *cfg, const double *moments, const double *com_off, double *L, double *Lcorr);
int octo_fmm_static_status(int device);

/* ---- complete uniform-grid solve ------------------------------------
 * "The multipoles of each cell are composed of the multipoles of its child cells ... The expansion of
 * each cell is composed of the expansion due to its interactions with other cells at the same level, and
 * the expansion of its parent cell".  On an isolated (L321) cubic grid of n^3 leaf cells,
 * n a power of two >= 16: the leaves are point masses at their cell centres; parent multipoles (order 3,
 * about the centre of mass) come from their children (M2M) up to the level of 2^3 cells; every multipole
 * level runs the interaction step above (Eq. 15 list, correction optional) and receives its parent's
 * expansion (L2L); a leaf gets its parent's expansion evaluated at its centre plus the monopole sum over
 * every other leaf whose parent is not well separated from its own (Eq. 15 list + near field).
 * out = [4][n][n][n] = (phi, g_x, g_y, g_z), g = -(grad phi + correction); a cell's own mass contributes
 * nothing.  Same ownership rules as above: the caller lends the workspace, everything is enqueued on
 * cfg.stream, nothing is allocated.  Formulas: DESIGN.md section 12. */
typedef struct octo_fmm_solver octo_fmm_solver_t;
typedef struct {
    int n;                  /* leaf cells per axis, a power of two, 16 <= n <= 2048                     */
    double h;               /* leaf cell width                                                          */
    double theta;           /* opening angle, 1/3 < theta < 1                                           */
    int am_correction;      /* 0/1: angular-momentum correction at the multipole levels (L127)          */
    int device;             /* CUDA device ordinal                                                      */
    void *stream;           /* cudaStream_t, borrowed                                                   */
    void *workspace;        /* device memory, 256-byte aligned, borrowed for the handle's lifetime      */
    size_t workspace_bytes; /* >= octo_fmm_solver_workspace_bytes(cfg)                                  */
    int two_rhs;            /* 1: also hold the per-level buffers of the second right-hand side, for
                               octo_fmm_solver_solve2 (about 1.6x the workspace); 0 otherwise              */
} octo_fmm_solver_config;

size_t octo_fmm_solver_workspace_bytes(const octo_fmm_solver_config *cfg);   /* 0 on invalid configuration */
int octo_fmm_solver_create(const octo_fmm_solver_config *cfg, octo_fmm_solver_t **out);
/* mass: device, [n][n][n] (x fastest); out: device, [4][n][n][n]; both 16-byte aligned (else EINVAL).
 * Asynchronous on the stream. */
int octo_fmm_solver_solve(octo_fmm_solver_t *s, const double *mass, double *out);
/* Second right-hand side (Alg. 1: "Compute g, phi, and d(phi)/dt using the
 * FMM ... with the numerically computed value of d(rho)/dt as the source term").  dmass: device, [n][n][n], the
 * time derivative of the cell masses (any sign); dphi_dt: device, [n][n][n] (only the potential of this solve is
 * used, Eq. 3; both 16-byte aligned).
 * Same tree, lists, kernels and EXPANSION CENTRES as the last octo_fmm_solver_solve() on this handle (the centres
 * of mass of the density, kept in the workspace; ESTATE if there was none), no angular-momentum correction (it
 * belongs to the force, L127), all dipole terms evaluated (the sources are not expanded about their own centres).
 * Asynchronous on the stream; overwrites the per-level results of solve().  At the multipole levels the two
 * right-hand sides share the geometry, not the pair arithmetic (DESIGN.md section 10a says why a fused kernel was
 * not built); the leaf sum is a potential-only tensor-core contraction over the 8 children of a parent. */
int octo_fmm_solver_solve_rhs2(octo_fmm_solver_t *s, const double *dmass, double *dphi_dt);
/* Both right-hand sides in ONE call (Alg. 1: "Compute g, phi, and d(phi)/dt using the FMM"): out as
 * octo_fmm_solver_solve, dphi_dt as octo_fmm_solver_solve_rhs2 (same readings: the centres of the density, no correction
 * for the second).  One upward pass builds both sets of multipoles, one downward pass stages both at every level; on the
 * levels that run one warp per cell the two share ONE launch (list walk, separation, 1/r, radial factors); on the finer
 * levels each runs the slab-fed kernel on its own sources (a fused kernel there is selectable with
 * octo_fmm_solver_set_option(s, "f2_fused", 1); measured slower).  Needs cfg.two_rhs = 1 (ESTATE
 * otherwise).  All four arrays device, 16-byte aligned.  Asynchronous on the stream. */
int octo_fmm_solver_solve2(octo_fmm_solver_t *s, const double *mass, const double *dmass, double *out, double *dphi_dt);
/* "f2_fused": 0 (default) | 1, see above.  "kernel": 0 (default) | 1 -- the slab-fed or the direct interaction kernel on
 * the levels that do not run one warp per cell (cross-check and measurement; same numbers to round-off). */
int octo_fmm_solver_set_option(octo_fmm_solver_t *s, const char *key, int value);
/* The same with HOST buffers: H2D of the masses into scratch, solve, D2H of out, stream synchronise.
 * scratch: device, >= octo_fmm_solver_host_scratch_bytes(cfg), borrowed for the call. */
size_t octo_fmm_solver_host_scratch_bytes(const octo_fmm_solver_config *cfg);
int octo_fmm_solver_solve_host(octo_fmm_solver_t *s, const double *mass_host, double *out_host, void *scratch,
                               size_t scratch_bytes);
/* Synchronises the stream; OCTO_FMM_EMASS if the correction met a cell of mass <= 0 at some level. */
int octo_fmm_solver_status(octo_fmm_solver_t *s);
int octo_fmm_solver_destroy(octo_fmm_solver_t *s);
/* Ordered in-domain pairs one solve evaluates, all levels. */
int octo_fmm_solver_interaction_count(const octo_fmm_solver_t *s, unsigned long long *n);
/* ... of which at the leaf level (monopole pairs, 8 flop each; the rest are multipole pairs). */
int octo_fmm_solver_leaf_interaction_count(const octo_fmm_solver_t *s, unsigned long long *n);
/* The leaf-level list (Eq. 15 list + near field) of a parity class, as octo_fmm_get_stencil. */
int octo_fmm_solver_get_leaf_stencil(const octo_fmm_solver_t *s, int parity, int *count, signed char (*dxyz)[3]);
/* Number of multipole levels (n/2 ... 2) and of kernels one solve launches. */
int octo_fmm_solver_num_levels(const octo_fmm_solver_t *s, int *multipole_levels, int *launches_per_solve);

/* ---- the solve on an ADAPTIVE oct-tree of 8^3 sub-grids -------------------------
 * "The FMM adapts naturally to an oct-tree based adaptive mesh refinement"; a node "is either
 * fully refined with eight child nodes (an interior node) or not refined at all (a leaf node)" and the mesh is
 * properly nested, so that a refinement boundary involves exactly two levels (L287-291).  The paper does not
 * describe the gravity side of such a boundary; the reading taken (R9) applies the rule of
 * L135 as a symmetric dual descent: a pair of one level whose parents are not well separated
 *   - is well separated (Eq. 15): interacts on that level with the general pair formula, whatever the kinds of
 *     the two cells (a leaf is the point mass M0 = m, M1 = M2 = M3 = 0, delta = 0; two leaves: the point-mass sum);
 *   - is not, both refined: left to the children;  both leaves: point masses, directly;
 *   - is not, A leaf and B refined: A meets the eight CHILDREN of B -- leaves one level down by proper nesting --
 *     as point masses, in both directions:  x_A - x_b = ((double)(2 i_A - i_b) + 0.5) * (h_A / 2) per axis.
 * Every pair is taken once in each direction with antisymmetric forces: linear momentum, and with the correction
 * angular momentum, are conserved as on a uniform grid (L125, L127); a fully refined tree IS the uniform solve.
 *
 * Layout: tree level l = 0 .. depth-1 lives on the lattice of n_l = n0 2^l cells per axis, h_l = h0 / 2^l.  Its arrays
 * cover a BOX of that lattice, box[6 l ..] = (lo_x, lo_y, lo_z, n_x, n_y, n_z) in cells of level l, all multiples of 8,
 * n >= 8, inside the lattice; box = NULL: every level is its whole lattice.  Level 0 must be the whole lattice.  Cells
 * outside a level's box do not exist on that level, so a deep tree costs memory and passes in proportion to the boxes,
 * not to the lattices (the paper's 9 levels, L684: a 2048^3 lattice with a box of a few hundred cells around a star).
 * Arrays are [n_z][n_y][n_x] of the box, x fastest.
 * kind[l] (uint8, HOST memory, read at create() only): 0 the cell does not exist on this level, 1 leaf, 2 refined;
 * constant over every aligned 8^3 sub-grid; every cell of level 0 exists; a cell exists on level l+1 iff its parent
 * is refined (so the 8 child sub-grids of a refined sub-grid lie inside the next box); no refined cell on the last
 * level (else EINVAL).  Proper nesting over the 26 neighbours of a sub-grid is the caller's duty (a leaf next to a
 * sub-grid two levels finer is not detected).  Above level 0 the uniform levels n0/2 .. 2 are built by the library.
 * mass[l]: DEVICE [box cells], read at the leaf cells only; out[l]: DEVICE [4][box cells] = (phi, g_x, g_y, g_z) at
 * the leaf cells, zeros elsewhere.  mass and out are HOST arrays of `depth` device pointers, all 16-byte aligned.
 * The caller lends the workspace.  create() uploads the topology from pageable memory and writes what no solve changes
 * (the zeros and the kind of every cell that is not refined, in the levels' moment arrays and staged records) on a stream
 * of the library's own, and synchronises it once.  A solve runs on streams of the library's own (its levels side by side),
 * behind whatever cfg.stream held at the call, and cfg.stream waits for it: to the caller it is asynchronous work on
 * cfg.stream.  One handle is not thread-safe. */
typedef struct octo_fmm_tree octo_fmm_tree_t;
typedef struct {
    int n0;                 /* cells per axis of level 0: a power of two, 8 <= n0 <= 2048                      */
    int depth;              /* number of tree levels, 1..12 (lattice of the last level <= 2^20 cells per axis;  */
                            /* every box <= 4096 cells per axis)                                               */
    double h0;              /* cell width of level 0                                                           */
    double theta;           /* opening angle, 1/3 < theta < 1                                                  */
    int am_correction;      /* 0/1 (L127)                                                                      */
    int device;
    void *stream;           /* cudaStream_t, borrowed                                                          */
    void *workspace;        /* device memory, 256-byte aligned, borrowed for the handle's lifetime             */
    size_t workspace_bytes; /* >= octo_fmm_tree_workspace_bytes(cfg, kind_host, box)                           */
} octo_fmm_tree_config;

size_t octo_fmm_tree_workspace_bytes(const octo_fmm_tree_config *cfg, const unsigned char *const *kind_host,
                                     const int *box);                                              /* 0 if invalid */
int octo_fmm_tree_create(const octo_fmm_tree_config *cfg, const unsigned char *const *kind_host, const int *box,
                         octo_fmm_tree_t **out);
/* Asynchronous on the stream. */
int octo_fmm_tree_solve(octo_fmm_tree_t *t, const double *const *mass, double *const *out);
/* Second right-hand side on the tree (L81-83, Alg. 1): dmass[l] DEVICE [box cells], the time derivative of the leaf
 * masses (any sign); dphi_dt[l] DEVICE [box cells]: the potential of these sources at the leaf cells, zeros elsewhere
 * (only the potential of this solve is used, Eq. 3).  Same tree, lists and EXPANSION CENTRES as the last
 * octo_fmm_tree_solve on this handle (ESTATE if there was none), no angular-momentum correction.  Overwrites the
 * per-level results of solve().  Asynchronous on the stream. */
int octo_fmm_tree_solve_rhs2(octo_fmm_tree_t *t, const double *const *dmass, double *const *dphi_dt);
/* The same solve, and the ordered pairs it evaluates, counted on the device for the bit-exact check of the pair set:
 * counts[0] multipole pairs of all levels (uniform levels included), counts[1] leaf-leaf point-mass pairs of one
 * level, counts[2] point-mass pairs across a refinement boundary.  Synchronises the stream. */
int octo_fmm_tree_interaction_counts(octo_fmm_tree_t *t, const double *const *mass, double *const *out,
                                     unsigned long long counts[3]);
/* The same with HOST buffers (mass_host[l], out_host[l]: host arrays of the layouts above; pinned memory makes the
 * copies asynchronous): H2D of the masses of every level that has leaves, solve, D2H of every out[l]; the copies
 * overlap the solve (masses arrive deepest level first on the streams that read them, a level's output leaves as soon
 * as its leaves are finished).  Returns when every out_host[l] is complete (synchronises the library's streams, not the
 * caller's).  scratch: device, >= octo_fmm_tree_host_scratch_bytes(t), 256-byte aligned, borrowed for the call. */
size_t octo_fmm_tree_host_scratch_bytes(const octo_fmm_tree_t *t);
int octo_fmm_tree_solve_host(octo_fmm_tree_t *t, const double *const *mass_host, double *const *out_host, void *scratch,
                             size_t scratch_bytes);
/* Synchronises the stream; OCTO_FMM_EMASS if the correction met an existing cell of mass <= 0. */
int octo_fmm_tree_status(octo_fmm_tree_t *t);
/* Kernels one solve launches. */
int octo_fmm_tree_launches(const octo_fmm_tree_t *t, int *launches);
int octo_fmm_tree_destroy(octo_fmm_tree_t *t);

#ifdef __cplusplus
}
#endif
#endif /* OCTO_FMM_H */
