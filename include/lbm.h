/*
 * lbm.h -- C ABI of the B200-native fused lattice Boltzmann stream-and-collide library
 *          (liblbm_b200.so, sm_100a).  Method: arXiv 1311.2404 (Sailfish); P:<n> cites line n
 *          of PAPER.md, A<n> cites a reading listed in DESIGN.md.
 *
 * Conventions (all calls)
 *   - Return value: 0 = LBM_OK, < 0 = error code below.  Nothing throws, nothing aborts.
 *     lbm_last_error(ctx) gives a human-readable string for the last failure on that context
 *     (ctx == NULL: the last failure of lbm_workspace_bytes / lbm_create on this thread).
 *   - Every pointer named d_* is a DEVICE pointer, every pointer named h_* is a HOST pointer.
 *     The caller owns all memory, including the workspace: the library never allocates device
 *     memory (the caller, e.g. PyTorch, allocates it and provides the stream).
 *   - Arrays are C-order [z][y][x], x fastest.  `real` is float (LBM_F32) or double
 *     (LBM_F64).  Scalar fields: real[nz][ny][nx].  Velocity: real[D][nz][ny][nx] (component
 *     planes, D = 2 for D2Q9, 3 for D3Q19).  Distributions: real[Q][nz][ny][nx] in the velocity
 *     order of reading A2 (lbm_lattice_info returns it).
 *   - The lattice is a torus: every axis is periodic.  Walls exist only through the
 *     node-type mask (LBM_NODE_*): SOLID nodes are dry and reflect by half-way bounce-back
 *     (reading A8); WALL_FULLWAY and VELOCITY nodes are described at the enum below.
 *   - All work is enqueued on the CUDA stream given to lbm_create; calls are asynchronous with
 *     respect to the host unless stated otherwise.  A context is not thread-safe.
 *   - `comp` is 0 except for LBM_SC2 (0 = component A, 1 = component B).
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { LBM_OK = 0, LBM_EINVAL = -1, LBM_EUNSUPPORTED = -2, LBM_ENOMEM = -3, LBM_ECUDA = -4, LBM_ESTATE = -5 };
enum { LBM_D2Q9 = 0, LBM_D3Q19 = 1 };            /* lattice, Table 1              */
enum { LBM_BGK = 0, LBM_MRT = 1, LBM_SC2 = 2,    /* model: SC2 = two LBGK components coupled
                                                    by the Shan-Chen force       */
       LBM_BGK_REG = 3,                          /* regularized LBGK (reading A23)    */
       LBM_BGK_LES = 4 };                        /* LBGK + Smagorinsky subgrid model, eq. (8)-(9) */
enum { LBM_F32 = 0, LBM_F64 = 1 };               /* precision of storage and arithmetic      */
enum { LBM_PSI_RHO = 0, LBM_PSI_1MEXP = 1 };     /* psi(rho) = rho | 1 - exp(-rho)   */
enum { LBM_STORE_AB = 0, LBM_STORE_AA = 1 };     /* two copies | in-place AA */
enum { LBM_FORCE_GUO = 0, LBM_FORCE_EDM = 1 };   /* Guo, eq. (17) P:251 | Exact Difference Method,
                                                    eq. (18), reading A22            */
/* node types of the lbm_set_geometry mask (P:446 reduced to what the path needs):
 *   FLUID         wet, collides
 *   SOLID         dry; a pull from it returns the puller's own opposite post-collision population
 *                 in the same step (half-way bounce-back, reading A8)
 *   WALL_FULLWAY  dry; stores the populations streamed into it and scatters them back reversed,
 *                 without relaxation, so they return one step later (full-way bounce-back,
 *                 Fig. 2 (1), reading A20)
 *   VELOCITY      wet; post-collision state f^eq(rho, bc_velocity) with rho from its own incoming
 *                 populations, missing ones = bounce-back copies, i.e. put a SOLID node behind it
 *                 (equilibrium velocity boundary, reading A21)
 * Any other byte value is SOLID. */
enum { LBM_NODE_FLUID = 0, LBM_NODE_SOLID = 1, LBM_NODE_WALL_FULLWAY = 2, LBM_NODE_VELOCITY = 3 };

#define LBM_QMAX 19

typedef struct lbm_ctx lbm_ctx;

typedef struct {
    uint32_t struct_size;     /* = sizeof(lbm_params); lets the ABI grow                           */
    int32_t lattice;          /* LBM_D2Q9 | LBM_D3Q19                                              */
    int32_t model;            /* LBM_BGK | LBM_MRT | LBM_SC2 | LBM_BGK_REG | LBM_BGK_LES          */
    int32_t precision;        /* LBM_F32 | LBM_F64                                                 */
    int32_t nx, ny, nz;       /* lattice extents, each >= 1 (nz == 1 for D2Q9), ny and nz <= 65535,
                                 nx*ny*nz <= 2^31 - 512                                            */
    double tau[2];            /* BGK/MRT: tau[0] > 0.5.  SC2: tau[0] = tau_A, tau[1] = tau_B       */
    double rates[LBM_QMAX];   /* MRT: Q relaxation rates in the moment order of reading A5;
                                 each in [0, 2]; ignored by the other models (eq. 4)        */
    double force[3];          /* body acceleration g; force density F = rho g (eq. 16, reading A4) */
    double sc_G;              /* Shan-Chen coupling G of eq. (10), sign per reading A11    */
    int32_t sc_psi;           /* LBM_PSI_*                                                         */
    int32_t store;            /* LBM_STORE_AB (default 0) | LBM_STORE_AA                           */
    double bc_velocity[3];    /* velocity imposed on LBM_NODE_VELOCITY nodes (reading A21);
                                 each component within (-1, 1); callers built against the 240-byte
                                 struct (no such field) get 0                                      */
    int32_t force_scheme;     /* LBM_FORCE_GUO (default 0, eq. 17) | LBM_FORCE_EDM (eq. 18); applies to
                                 the body force and to the Shan-Chen coupling force alike          */
    int32_t reserved_;        /* keeps sizeof a multiple of 8; must be 0 (LBM_EINVAL otherwise)    */
    double smagorinsky_cs;    /* LBM_BGK_LES: Smagorinsky constant C_S of eq. (9) (0.1), in [0, 10) */
} lbm_params;

/* Static description of a lattice (Table 1; ordering = reading A2).
 * e: int32[Q][3], w: double[Q], opp: int32[Q] (index of -e_i); any may be NULL.
 * Writes Q and D.  Host pointers.  LBM_EINVAL on an unknown lattice. */
int lbm_lattice_info(int32_t lattice, int32_t *Q, int32_t *D, int32_t *h_e, double *h_w, int32_t *h_opp);

/* Bytes of device workspace a context with these parameters needs (distribution store,
 * node-type/link encoding, Shan-Chen fields, staging for the host-buffer calls). */
int lbm_workspace_bytes(const lbm_params *p, size_t *bytes);

/* Create a context on the current CUDA device.  d_workspace: >= lbm_workspace_bytes, 256-byte
 * aligned, owned by the caller and kept alive until lbm_destroy.  cuda_stream: a cudaStream_t
 * (NULL = legacy default stream).  The geometry starts all-FLUID.
 * Errors: LBM_EINVAL (bad enum/size/tau/rate, workspace too small or misaligned),
 * LBM_EUNSUPPORTED (combination not built, e.g. MRT on SC2), LBM_ECUDA. */
int lbm_create(const lbm_params *p, void *d_workspace, size_t bytes, void *cuda_stream, lbm_ctx **out);
int lbm_destroy(lbm_ctx *ctx);

/* Node types.  d_mask: uint8[nz][ny][nx] of LBM_NODE_* values.  Builds the internal link
 * encoding (which of the Q pull sources are reflected).  Must be called before lbm_init_equilibrium /
 * lbm_set_distributions if the geometry is not all-FLUID; calling it afterwards returns LBM_ESTATE.
 * SYNCHRONISES the stream once: it reads back how many nodes touch a wall to pick the kernel variant
 * (lbm_get_dispatch reports the choice), so that lbm_step never has to block. */
int lbm_set_geometry(lbm_ctx *ctx, const uint8_t *d_mask);
int lbm_get_geometry(lbm_ctx *ctx, uint8_t *d_mask);          /* writes LBM_NODE_* per node */

/* f_i(x, 0) = f_i^eq(rho0(x), u0(x)), eq. (3), velocity used as given (A15).
 * d_rho: real[N], d_u: real[D][N].  SOLID nodes are ignored. */
int lbm_init_equilibrium(lbm_ctx *ctx, int comp, const void *d_rho, const void *d_u);

/* Advance n >= 0 time steps; each step is one fused pull-stream + moments + equilibrium +
 * collision (+ Guo source) + store pass over the lattice (Alg. 1; eqs. 1-4, 16-17);
 * LBM_SC2 runs the macro-field pass and then the coupled collide pass (eq. 10).
 * LBM_ESTATE if a component has not been initialised.  Asynchronous: never blocks the host.
 * Lattices of up to 2^20 nodes replay 50-step CUDA graphs (captured on a private stream at the first
 * call that needs them); single-component AB lattices of up to 4096 nodes (D2Q9: 16384) run all n steps
 * in one launch of a thread-block cluster that keeps the store in distributed shared memory, falling
 * back to the graph path where such a cluster cannot be scheduled; results are bit-identical to
 * single-step launches. */
int lbm_step(lbm_ctx *ctx, int n);

/* rho = sum_i f_i, velocity v of eq. (16) (includes g/2) from the current state.
 * SC2: rho_s and the bare component velocity j_s / rho_s.  Dry nodes (SOLID, WALL_FULLWAY): rho = 0, u = 0.
 * d_rho: real[N] or NULL, d_u: real[D][N] or NULL. */
int lbm_macro(lbm_ctx *ctx, int comp, void *d_rho, void *d_u);

/* Test / checkpoint hooks.  Canonical state = pre-collision, post-streaming f_i(x, t) (what
 * Alg. 1 line 4 loads; reading A9), real[Q][N].  get writes 0 on SOLID nodes; set ignores them. */
int lbm_get_distributions(lbm_ctx *ctx, int comp, void *d_f);
int lbm_set_distributions(lbm_ctx *ctx, int comp, const void *d_f);

/* Streaming index map (reading A8): d_map int64[Q][N]; map[i][x] = i' * N + x' = the slot of the
 * canonical post-collision array whose value becomes f_i(x, t+1): (i, x - e_i) unless that node is
 * SOLID (FLUID, WALL_FULLWAY and VELOCITY sources are pulled directly), else (ibar, x); -1 where x
 * is SOLID.  Computed by the same device routine the step kernels use for their gather. */
int lbm_get_stream_map(lbm_ctx *ctx, int64_t *d_map);

/* Whole path with HOST buffers (what bench.py's e2e leg times): H2D of mask, rho0, u0 per
 * component -> set_geometry -> init_equilibrium -> step(n) -> macro(comp 0) -> D2H, then
 * synchronises the stream.  h_mask may be NULL (all FLUID).  h_rho0 / h_u0: arrays of `ncomp`
 * host pointers.  h_rho_out / h_u_out (component 0) may be NULL.  Resets the context state. */
int lbm_run_host(lbm_ctx *ctx, const uint8_t *h_mask, const void *const *h_rho0, const void *const *h_u0,
                 int n, void *h_rho_out, void *h_u_out);

/* z-slab decomposition of one lattice over several contexts (section 3.6 of the paper).
 * Each slab is an ordinary context whose local lattice is its share of the global z-planes PLUS one ghost
 * plane below (local z = 0) and one above (local z = nz - 1): the caller slices mask, rho0 and u0 of the
 * global lattice accordingly (ghost planes = copies of the neighbour's boundary planes, through the
 * periodic seam if periodic_z) and initialises every slab with the usual calls.  lbm_step_slabs then
 * advances all slabs n steps in lockstep.  Every step launches the two boundary interior planes of each
 * slab first; as soon as they are done each ghost plane receives, from the neighbouring slab's boundary
 * plane, the 5 of 19 populations that stream across the face -- on a side stream, concurrently with
 * the launch over the bulk planes; ghost planes themselves are never updated.  For LBM_SC2 the
 * macro-field pass is ordered the same way and exchanges the psi planes before the collide pass.
 * slabs[0] is the lowest slab; periodic_z != 0 also links slabs[count-1] to slabs[0].  Interior planes
 * then hold exactly the bits of a single context running the whole lattice; ghost planes are scratch.
 * Contexts may use different streams (ordered by events) and, with peer access enabled, different
 * devices; D3Q19, AB store.  Errors: LBM_EINVAL (mismatching slabs), LBM_EUNSUPPORTED, LBM_ESTATE. */
int lbm_step_slabs(lbm_ctx *const *slabs, int count, int periodic_z, int n);

/* The path in one call that ALLOCATES NOTHING, for callers that can neither call cudaMalloc nor hand over a
 * workspace (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).  The
 * context's workspace lives in a file-scope device array of LBM_NOALLOC_MAX_BYTES inside the library (every
 * GPU that loads the library holds it until the process exits).  The call builds a context in that array,
 * runs lbm_set_geometry(d_mask) -> lbm_set_distributions(d_f_in) -> lbm_step(n) -> lbm_get_distributions
 * (d_f_out) on `cuda_stream` with the ordinary kernels, and destroys the context; it calls no cudaMalloc,
 * cudaFree, stream or graph creation.  p: as for lbm_create, LBM_STORE_AB only.  d_mask: uint8[N] or NULL (all
 * FLUID; with a mask the call synchronises the stream once, as lbm_set_geometry does).  d_f_in, d_f_out:
 * canonical distributions real[ncomp][Q][N] (LBM_SC2: component A then B), caller-owned device memory, may be
 * the same buffer.  Asynchronous otherwise.
 * Limits: lbm_workspace_bytes(p) <= LBM_NOALLOC_MAX_BYTES (D3Q19 fp32 up to 64^3 nodes), else LBM_EINVAL with
 * a message naming both sizes (lbm_noalloc_last_error).  ALL calls on a device share the one array, which
 * keeps the last call's contents (the call clears what must start at zero): calls are safe back to back on
 * one stream, but calls that overlap on the GPU (different streams, different threads) RACE. */
#define LBM_NOALLOC_MAX_BYTES (64u << 20)
int lbm_step_noalloc(const lbm_params *p, const uint8_t *d_mask, const void *d_f_in, void *d_f_out, int n,
                     void *cuda_stream);
const char *lbm_noalloc_last_error(void);   /* message of the last failed lbm_step_noalloc on this thread */

/* Time step counter since the last init/set, and number of kernels launched by this context. */
int lbm_get_counters(const lbm_ctx *ctx, int64_t *steps, int64_t *launches);

/* Which kernel variant lbm_step uses for this context (chosen from the lattice size at lbm_create and
 * from the geometry at lbm_set_geometry).  For tests and benchmarks that must
 * state what they measured. */
typedef struct {
    int32_t nodes_per_thread;        /* consecutive x-nodes per thread of the step kernels: 1, 2 or 4 */
    int32_t index_bits;              /* 32 or 64: width of slot indices i * N + node                  */
    int32_t graph_replay;            /* > 0: steps per replayed CUDA graph (small lattices), else 0   */
    int32_t resident_nodes_per_cta;  /* > 0: cluster-resident path, nodes per CTA                     */
    int32_t resident_ctas;           /* CTAs of that cluster (8 or 16), else 0                        */
    int32_t rows_per_block;          /* > 0: row-walking kernel for obstacle-rich geometries          */
    int32_t block_threads;           /* threads per block of the step kernels                         */
    int32_t sc_split;                /* LBM_SC2: 1 = one collide launch per component, 0 = one
                                        launch for both                                               */
    int32_t rows_strided;            /* row-walking kernel: 1 = a thread's two nodes lie half a row apart (2 nodes per thread) */
} lbm_dispatch;
int lbm_get_dispatch(const lbm_ctx *ctx, lbm_dispatch *out);

/* Test-only tuning knobs.  Environment variables, read at lbm_create / lbm_set_geometry and honoured
 * ONLY if LBM_TUNING=1 is set too: LBM_VEC (1|2|4 nodes per thread), LBM_IDX64 (1: 64-bit slot indices),
 * LBM_BLOCK_X, LBM_BLOCK_THREADS (multiples of 32), LBM_ROWS (rows per block of the row-walking kernel,
 * 0 = off), LBM_ROWS_STRIDED, LBM_NO_GRAPH, LBM_NO_RESIDENT, LBM_RESIDENT_MAX (largest lattice of the cluster-resident
 * path), LBM_SC_SPLIT (0: monolithic two-component collide kernel), LBM_SC_FIELDS_VEC, LBM_SPAN_BX.  They select among kernels that all pass the same parity tests; they are not part of the ABI. */

const char *lbm_last_error(const lbm_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
