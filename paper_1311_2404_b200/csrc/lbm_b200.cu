// lbm_b200.cu -- the C ABI of include/lbm.h: argument checking, workspace carving, graph replay.
// All arithmetic of the method lives in the kernels (lbm_kernels.cuh / lbm_node.cuh), dispatched
// through lbm_impl.cuh; nothing here touches oracle/.
#include "lbm_impl.cuh"

namespace {

// sizeof(lbm_params) before bc_velocity was appended; such callers get bc_velocity = 0
constexpr uint32_t LBM_PARAMS_SIZE_V1 = 240;
// ... and before force_scheme was appended; such callers get the Guo scheme
constexpr uint32_t LBM_PARAMS_SIZE_V2 = 264;
// ... and before smagorinsky_cs was appended
constexpr uint32_t LBM_PARAMS_SIZE_V3 = 272;

int validate(const lbm_params *p, int *Q, int *D) {
    if (!p) return fail(nullptr, LBM_EINVAL, "params is NULL");
    if (p->struct_size != sizeof(lbm_params) && p->struct_size != LBM_PARAMS_SIZE_V1 && p->struct_size != LBM_PARAMS_SIZE_V2 &&
        p->struct_size != LBM_PARAMS_SIZE_V3)
        return fail(nullptr, LBM_EINVAL, "struct_size is not a known sizeof(lbm_params)");
    if (p->lattice != LBM_D2Q9 && p->lattice != LBM_D3Q19) return fail(nullptr, LBM_EINVAL, "unknown lattice");
    if (p->model < LBM_BGK || p->model > LBM_BGK_LES) return fail(nullptr, LBM_EINVAL, "unknown model");
    if (p->precision != LBM_F32 && p->precision != LBM_F64) return fail(nullptr, LBM_EINVAL, "unknown precision");
    if (p->store != LBM_STORE_AB && p->store != LBM_STORE_AA) return fail(nullptr, LBM_EINVAL, "unknown store");
    if (p->nx < 1 || p->ny < 1 || p->nz < 1) return fail(nullptr, LBM_EINVAL, "extents must be >= 1");
    if (p->lattice == LBM_D2Q9 && p->nz != 1) return fail(nullptr, LBM_EINVAL, "D2Q9 needs nz == 1");
    // node indices are ints and padded threads index up to one block beyond the last node
    if ((double)p->nx * p->ny * p->nz > 2147483648.0 - 512.0) return fail(nullptr, LBM_EINVAL, "nx*ny*nz must be <= 2^31 - 512");
    if (p->struct_size >= LBM_PARAMS_SIZE_V3 && p->reserved_ != 0) return fail(nullptr, LBM_EINVAL, "reserved_ must be 0");
    const int nt = p->model == LBM_SC2 ? 2 : 1;
    for (int s = 0; s < nt; s++)
        if (!(p->tau[s] > 0.5)) return fail(nullptr, LBM_EINVAL, "tau must be > 0.5");
    *Q = p->lattice == LBM_D2Q9 ? 9 : 19;
    *D = p->lattice == LBM_D2Q9 ? 2 : 3;
    if (p->model == LBM_MRT)
        for (int k = 0; k < *Q; k++)
            if (!(p->rates[k] >= 0.0 && p->rates[k] <= 2.0)) return fail(nullptr, LBM_EINVAL, "MRT rates must be in [0, 2]");
    for (int a = 0; a < 3; a++)
        if (!(p->force[a] == p->force[a])) return fail(nullptr, LBM_EINVAL, "force is NaN");
    if (p->model == LBM_BGK_LES && (p->struct_size != sizeof(lbm_params) || !(p->smagorinsky_cs >= 0.0 && p->smagorinsky_cs < 10.0)))
        return fail(nullptr, LBM_EINVAL, "LBM_BGK_LES needs smagorinsky_cs in [0, 10)");
    if (p->model == LBM_BGK_REG && (p->struct_size < LBM_PARAMS_SIZE_V3 || p->force_scheme != LBM_FORCE_EDM) &&
        (p->force[0] != 0.0 || p->force[1] != 0.0 || p->force[2] != 0.0))
        return fail(nullptr, LBM_EUNSUPPORTED, "regularized LBGK takes a body force through LBM_FORCE_EDM only (reading A23)");
    if (p->struct_size >= LBM_PARAMS_SIZE_V3 && p->force_scheme != LBM_FORCE_GUO && p->force_scheme != LBM_FORCE_EDM)
        return fail(nullptr, LBM_EINVAL, "unknown force_scheme");
    if (p->struct_size >= LBM_PARAMS_SIZE_V2)
        for (int a = 0; a < 3; a++)
            if (!(p->bc_velocity[a] > -1.0 && p->bc_velocity[a] < 1.0)) return fail(nullptr, LBM_EINVAL, "bc_velocity must be within (-1, 1)");
    if (p->model == LBM_SC2 && p->sc_psi != LBM_PSI_RHO && p->sc_psi != LBM_PSI_1MEXP)
        return fail(nullptr, LBM_EINVAL, "unknown sc_psi");
    if (p->lattice == LBM_D2Q9 && p->force[2] != 0.0) return fail(nullptr, LBM_EINVAL, "D2Q9 force has no z component");
    if (p->ny > 65535 || p->nz > 65535) return fail(nullptr, LBM_EUNSUPPORTED, "ny and nz must be <= 65535");
    return LBM_OK;
}

void make_layout(const lbm_params *p, int Q, int D, Layout *L) {
    const size_t N = (size_t)p->nx * p->ny * p->nz, rs = p->precision == LBM_F32 ? 4 : 8;
    const int nc = p->model == LBM_SC2 ? 2 : 1;
    size_t off = 0;
    memset(L, 0, sizeof *L);
    for (int s = 0; s < nc; s++)
        for (int b = 0; b < 2; b++) {
            if (b == 1 && p->store == LBM_STORE_AA) { L->store[s][1] = L->store[s][0]; continue; }  // in place
            L->store[s][b] = off; off += align_up(Q * N * rs);
        }
    L->type = off; off += align_up(N);
    L->link = off; off += align_up(4 * N);
    L->counters = off; off += ALIGN;
    if (nc == 2)
    {   // (psi_A, psi_B) interleaved, or planar psi_A | psi_B for the split kernels; u' of the split kernels
        L->psi[0] = L->psi[1] = off; off += align_up(2 * N * rs);
        L->up = off; off += align_up((size_t)D * N * rs);
    }
    L->stage_mask = off; off += align_up(N);
    L->stage_rho = off; off += align_up(N * rs);
    L->stage_u = off; off += align_up(D * N * rs);
    L->total = off;
}

const Vtbl *select_impl(const lbm_params *p) {
    const void *t = p->lattice == LBM_D2Q9 ? (p->precision == LBM_F32 ? lbm_impl_d2q9_f32() : lbm_impl_d2q9_f64())
                                           : (p->precision == LBM_F32 ? lbm_impl_d3q19_f32() : lbm_impl_d3q19_f64());
    return static_cast<const Vtbl *>(t);
}

// Test-only tuning knobs (include/lbm.h lists them): honoured only when LBM_TUNING=1 is set as well,
// so that a stray variable in a user's environment cannot change the kernel selection.
bool tuning_enabled() {
    const char *e = getenv("LBM_TUNING");
    return e && e[0] == '1' && e[1] == 0;
}

int env_int(const char *name, int dflt, int lo, int hi) {
    if (!tuning_enabled()) return dflt;
    if (const char *e = getenv(name)) {
        const int v = atoi(e);
        if (v >= lo && v <= hi) return v;
    }
    return dflt;
}

// Nodes per thread of the step kernels, by measurement (profiles/):
//   fp32 single component: 4-node packs (16-byte accesses) on mostly-bulk geometries (c2: 44.1 vs
//   39.7 GLUPS at V = 1); 2-node packs when many nodes are BOUNDARY, where the reflected-link
//   fix-up of 4 nodes costs too many registers (c3: V = 2 34.8, V = 4 29.5, V = 1 26.1 GLUPS);
//   fp64: 2-node packs (c4: 22.4 vs 22.1); two-component kernel: register-bound, 1 node (c5: 12.0 vs 9.9).
// LBM_VEC overrides (tuning knob, not part of the ABI).  Falls back to what divides nx.
int pick_vec(const lbm_params *p, double nonbulk_fraction, bool sc_split = false) {
    const int widest = p->precision == LBM_F32 ? 4 : 2;
    int v = 1;
    if (p->model != LBM_SC2 || sc_split) v = p->precision == LBM_F64 ? 2 : (nonbulk_fraction < 0.2 ? 4 : 2);
    // regularized LBGK / Smagorinsky carry six second moments per node: 2-node packs (cavity box:
    // LES 43.0 vs 33.9 GLUPS at V = 4, regularized 42.9 vs 41.4)
    // and so does MRT with its 19 moments (cavity box: 43.0 vs 41.0 GLUPS)
    if (p->model == LBM_BGK_REG || p->model == LBM_BGK_LES || p->model == LBM_MRT) v = v > 2 ? 2 : v;
    // small lattices cannot fill 148 SMs with wide packs (us per step at V = 1/2/4: D2Q9 128^2 1.68/1.83/2.14,
    // 256^2 2.07/2.14/2.35, 512^2 3.46/3.20/3.67; D3Q19 48^3 3.86/3.53/4.92, 64^3 5.73/5.61/8.03, 96^3 23.3/22.2/23.3)
    const int64_t sites = (int64_t)p->nx * p->ny * p->nz;
    if (sites <= (1 << 16)) v = 1;
    else if (sites < (1 << 20) && v > 2) v = 2;
    v = env_int("LBM_VEC", v, 1, widest);
    if (v == 3) v = 2;
    // MRT, regularized LBGK and Smagorinsky lose at V = 4 (above): those kernels are not built (a quarter of the build)
    if (!sc_split && p->model != LBM_BGK && p->model != LBM_SC2 && v > 2) v = 2;
    while (v > 1 && p->nx % v) v /= 2;
    return v;
}

// Cluster-resident path (resident_kernel): single component, AB store, one node per thread, both
// buffers of a CTA's share of the lattice in its shared memory.  8 CTAs x 512 nodes up to 4096 nodes;
// D2Q9 also 16 CTAs (non-portable cluster size) x 512 / 1024 nodes up to 16384 nodes (c1: 128^2).
int pick_resident(const lbm_params *p, int Q, int64_t N, int *ctas) {
    if (p->model == LBM_SC2 || p->store != LBM_STORE_AB || env_int("LBM_NO_RESIDENT", 0, 0, 1)) return 0;
    const size_t rs = p->precision == LBM_F32 ? 4 : 8;
    const int64_t limit = env_int("LBM_RESIDENT_MAX", Q == 9 ? 16384 : 4096, 0, 16384);
    if (N > limit) return 0;
    *ctas = N <= 4096 ? 8 : RESIDENT_MAX_CTAS;
    int slog2 = 5;
    while (((int64_t)*ctas << slog2) < N) slog2++;
    const size_t S = (size_t)1 << slog2;
    if (S > (Q == 9 ? 1024u : 512u)) return 0;
    if (2 * (size_t)Q * S * rs > 200 * 1024) return 0;
    return slog2;
}

int pick_block_x(int nx) {
    const int forced = env_int("LBM_BLOCK_X", 0, 32, 256);
    if (forced && forced % 32 == 0) return forced;
    if (nx % 256 == 0) return 256;
    if (nx % 128 == 0) return 128;
    if (nx <= 256) return (nx + 31) / 32 * 32;
    return 128;
}

}  // namespace

// ---- exported C ABI ---------------------------------------------------------------------------
#define LBM_API extern "C" __attribute__((visibility("default")))
#define CHECK_CTX(c) do { if (!(c)) return fail(nullptr, LBM_EINVAL, "ctx is NULL"); } while (0)
#define CHECK_COMP(c, s) do { if ((s) < 0 || (s) >= (c)->ncomp) return fail((c), LBM_EINVAL, "comp out of range"); } while (0)

LBM_API int lbm_lattice_info(int32_t lattice, int32_t *Q, int32_t *D, int32_t *h_e, double *h_w, int32_t *h_opp) {
    auto fill = [&](auto Ltag) {
        using L = decltype(Ltag);
        if (Q) *Q = L::Q;
        if (D) *D = L::D;
        for (int i = 0; i < L::Q; i++) {
            if (h_e) { h_e[3 * i] = L::ex(i); h_e[3 * i + 1] = L::ey(i); h_e[3 * i + 2] = L::ez(i); }
            if (h_w) h_w[i] = L::template w<double>(i);
            if (h_opp) h_opp[i] = L::opp(i);
        }
    };
    if (lattice == LBM_D2Q9) fill(D2Q9{});
    else if (lattice == LBM_D3Q19) fill(D3Q19{});
    else return fail(nullptr, LBM_EINVAL, "unknown lattice");
    return LBM_OK;
}

LBM_API int lbm_workspace_bytes(const lbm_params *p, size_t *bytes) {
    int Q, D;
    if (int rc = validate(p, &Q, &D)) return rc;
    if (!bytes) return fail(nullptr, LBM_EINVAL, "bytes is NULL");
    Layout lay;
    make_layout(p, Q, D, &lay);
    *bytes = lay.total;
    return LBM_OK;
}

LBM_API int lbm_create(const lbm_params *p, void *d_workspace, size_t bytes, void *cuda_stream, lbm_ctx **out) {
    int Q, D;
    if (int rc = validate(p, &Q, &D)) return rc;
    if (!out) return fail(nullptr, LBM_EINVAL, "out is NULL");
    *out = nullptr;
    Layout lay;
    make_layout(p, Q, D, &lay);
    if (!d_workspace || bytes < lay.total) return fail(nullptr, LBM_EINVAL, "workspace NULL or smaller than lbm_workspace_bytes");
    if (reinterpret_cast<uintptr_t>(d_workspace) % ALIGN) return fail(nullptr, LBM_EINVAL, "workspace must be 256-byte aligned");
    lbm_ctx *c = new (std::nothrow) lbm_ctx();
    if (!c) return fail(nullptr, LBM_ENOMEM, "host allocation failed");
    memset(&c->p, 0, sizeof c->p);
    memcpy(&c->p, p, p->struct_size);  // a shorter (older) struct leaves the newer fields zero
    c->Q = Q; c->D = D; c->ncomp = p->model == LBM_SC2 ? 2 : 1;
    c->rs = p->precision == LBM_F32 ? 4 : 8;
    c->g.nx = p->nx; c->g.ny = p->ny; c->g.nz = p->nz; c->g.N = (int64_t)p->nx * p->ny * p->nz; c->g.z0 = 0;
    c->zsel0 = 0; c->zselc = p->nz; c->no_advance = false; c->slab_stream = nullptr; c->slab_event2 = nullptr;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    if (cudaGetDevice(&c->device) != cudaSuccess) { cudaGetLastError(); c->device = 0; }
    c->ws = static_cast<char *>(d_workspace);
    c->lay = lay;
    c->block_x = pick_block_x(p->nx);
    c->vec = pick_vec(p, 0.0);
    c->aa = p->store == LBM_STORE_AA;
    // slot numbers i * N + node: 32 bits whenever Q * N < 2^32; the 64-bit kernels exist for the AB store of
    // D3Q19 LBGK / MRT / (split) Shan-Chen, which is what a lattice of that size (> 226 M nodes) would run
    const bool idx64_built = p->lattice == LBM_D3Q19 && p->store == LBM_STORE_AB &&
                             (p->model == LBM_BGK || p->model == LBM_MRT || p->model == LBM_SC2);
    c->idx32 = (double)Q * (double)c->g.N < 4294967296.0;
    if (!c->idx32 && !idx64_built) {
        delete c;
        return fail(nullptr, LBM_EUNSUPPORTED, "Q*nx*ny*nz >= 2^32 is built for D3Q19 with the AB store and LBM_BGK / LBM_MRT / LBM_SC2 only");
    }
    if (idx64_built && env_int("LBM_IDX64", 0, 0, 1)) c->idx32 = false;
    c->rows = 0;
    c->rows_strided = 0;
    c->sc_phase = 0;
    c->slab_event = nullptr;
    c->sc_split = (p->model == LBM_SC2 && (env_int("LBM_SC_SPLIT", 1, 0, 1) || p->store == LBM_STORE_AA || !c->idx32)) ? pick_vec(p, 0.0, true) : 0;
    c->all_bulk = true;  // the geometry starts all-FLUID
    c->span_bx = env_int("LBM_SPAN_BX", 0, 32, 256) / 32 * 32;
    c->sc_fields_vec = env_int("LBM_SC_FIELDS_VEC", 1, 1, 2);
    if (p->nx % 2) c->sc_fields_vec = 1;
    c->block_threads = env_int("LBM_BLOCK_THREADS", 64, 32, 256) / 32 * 32;
    c->vt = select_impl(p);
    c->err[0] = 0;
    c->resident_ctas = 8;
    c->resident_state = 0;
    c->resident_slog2 = pick_resident(p, Q, c->g.N, &c->resident_ctas);
    c->no_graph = env_int("LBM_NO_GRAPH", 0, 0, 1) != 0;
    c->use_graph = c->resident_slog2 == 0 && c->g.N <= GRAPH_MAX_SITES;
    c->capture_stream = nullptr;  // created at the first capture
    // geometry starts all-FLUID: type = BULK, link = 0
    cudaError_t e = cudaMemsetAsync(c->ws + lay.type, 0, (size_t)c->g.N, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->ws + lay.link, 0, 4 * (size_t)c->g.N, c->stream);
    if (e != cudaSuccess) {
        fail(nullptr, LBM_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
        if (c->capture_stream) cudaStreamDestroy(c->capture_stream);
        delete c;
        return LBM_ECUDA;
    }
    *out = c;
    return LBM_OK;
}

LBM_API int lbm_destroy(lbm_ctx *c) {
    CHECK_CTX(c);
    drop_graphs(c);
    if (c->capture_stream) cudaStreamDestroy(c->capture_stream);
    if (c->slab_event) cudaEventDestroy(c->slab_event);
    if (c->slab_event2) cudaEventDestroy(c->slab_event2);
    if (c->slab_stream) cudaStreamDestroy(c->slab_stream);
    delete c;
    return LBM_OK;
}

LBM_API int lbm_set_geometry(lbm_ctx *c, const uint8_t *d_mask) {
    CHECK_CTX(c);
    if (!d_mask) return fail(c, LBM_EINVAL, "d_mask is NULL");
    if (c->geometry_frozen) return fail(c, LBM_ESTATE, "lbm_set_geometry after the state was initialised");
    if (int rc = c->vt->set_geometry(c, d_mask)) return rc;
    // How many nodes are not BULK decides the kernel variant (pack width; row-walking kernel for
    // obstacle-rich geometries).  Read it back here, once per geometry, so that lbm_step never blocks.
    unsigned nonbulk = 0;
    cudaError_t e = cudaMemcpyAsync(&nonbulk, c->ws + c->lay.counters, sizeof nonbulk, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return fail(c, LBM_ECUDA, "reading the geometry counter: %s", cudaGetErrorString(e));
    const double frac = (double)nonbulk / (double)c->g.N;
    c->all_bulk = nonbulk == 0;
    c->vec = pick_vec(&c->p, frac);
    if (c->sc_split) c->sc_split = pick_vec(&c->p, frac, true);
    c->rows = env_int("LBM_ROWS", frac >= 0.2 ? 2 : 0, 0, 65535);
    c->rows_strided = env_int("LBM_ROWS_STRIDED", 1, 0, 1);  // c3: 38.8 -> 39.6 GLUPS fp32, 20.0 -> 20.5 fp64 (20-step calls)
    return LBM_OK;
}

LBM_API int lbm_get_geometry(lbm_ctx *c, uint8_t *d_mask) {
    CHECK_CTX(c);
    if (!d_mask) return fail(c, LBM_EINVAL, "d_mask is NULL");
    get_geometry_kernel<<<grid_of(c), c->block_x, 0, c->stream>>>(c->g, at<uint8_t>(c, c->lay.type), d_mask);
    return check_launch(c, "get_geometry_kernel");
}

static void mark_initialised(lbm_ctx *c, int comp) {
    c->inited[comp] = true;
    c->geometry_frozen = true;
    c->steps = 0;
}

LBM_API int lbm_init_equilibrium(lbm_ctx *c, int comp, const void *d_rho, const void *d_u) {
    CHECK_CTX(c);
    CHECK_COMP(c, comp);
    if (!d_rho || !d_u) return fail(c, LBM_EINVAL, "d_rho / d_u is NULL");
    if (int rc = c->vt->init_equilibrium(c, comp, d_rho, d_u)) return rc;
    mark_initialised(c, comp);
    return LBM_OK;
}

LBM_API int lbm_set_distributions(lbm_ctx *c, int comp, const void *d_f) {
    CHECK_CTX(c);
    CHECK_COMP(c, comp);
    if (!d_f) return fail(c, LBM_EINVAL, "d_f is NULL");
    if (int rc = c->vt->set_distributions(c, comp, d_f)) return rc;
    mark_initialised(c, comp);
    return LBM_OK;
}

static int check_state(lbm_ctx *c) {
    for (int s = 0; s < c->ncomp; s++)
        if (!c->inited[s]) return fail(c, LBM_ESTATE, "a component has not been initialised");
    return LBM_OK;
}

LBM_API int lbm_step(lbm_ctx *c, int n) {
    CHECK_CTX(c);
    if (n < 0) return fail(c, LBM_EINVAL, "n < 0");
    if (int rc = check_state(c)) return rc;
    while (c->use_graph && !c->no_graph && n >= GRAPH_STEPS) {
        cudaGraphExec_t &exec = c->graph[c->cur];
        if (!exec) {  // capture GRAPH_STEPS ordinary step launches; nothing executes during capture
            if (!c->capture_stream && cudaStreamCreateWithFlags(&c->capture_stream, cudaStreamNonBlocking) != cudaSuccess) {
                cudaGetLastError();
                c->capture_stream = nullptr;
                c->no_graph = true;  // no private stream to capture on: plain launches
                break;
            }
            const int64_t steps0 = c->steps, launches0 = c->launches;
            const int cur0 = c->cur;
            const cudaStream_t user = c->stream;
            cudaGraph_t g = nullptr;
            cudaError_t e = cudaStreamBeginCapture(c->capture_stream, cudaStreamCaptureModeThreadLocal);
            if (e != cudaSuccess) return fail(c, LBM_ECUDA, "cudaStreamBeginCapture: %s", cudaGetErrorString(e));
            c->stream = c->capture_stream;
            const int rc = c->vt->step(c, GRAPH_STEPS);
            c->stream = user;
            e = cudaStreamEndCapture(c->capture_stream, &g);
            c->graph_launches = c->launches - launches0;
            c->steps = steps0;
            c->launches = launches0;
            c->cur = cur0;  // GRAPH_STEPS is even; a capture that failed half-way must not leave the parity flipped
            if (rc) { if (g) cudaGraphDestroy(g); return rc; }
            if (e == cudaSuccess) e = cudaGraphInstantiate(&exec, g, 0);
            if (g) cudaGraphDestroy(g);
            if (e != cudaSuccess) { exec = nullptr; return fail(c, LBM_ECUDA, "graph capture/instantiate: %s", cudaGetErrorString(e)); }
        }
        cudaError_t e = cudaGraphLaunch(exec, c->stream);
        if (e != cudaSuccess) return fail(c, LBM_ECUDA, "cudaGraphLaunch: %s", cudaGetErrorString(e));
        c->steps += GRAPH_STEPS;
        c->launches += c->graph_launches;
        n -= GRAPH_STEPS;
    }
    return c->vt->step(c, n);
}

LBM_API int lbm_macro(lbm_ctx *c, int comp, void *d_rho, void *d_u) {
    CHECK_CTX(c);
    CHECK_COMP(c, comp);
    if (!c->inited[comp]) return fail(c, LBM_ESTATE, "component has not been initialised");
    if (!d_rho && !d_u) return LBM_OK;
    return c->vt->macro(c, comp, d_rho, d_u);
}

LBM_API int lbm_get_distributions(lbm_ctx *c, int comp, void *d_f) {
    CHECK_CTX(c);
    CHECK_COMP(c, comp);
    if (!d_f) return fail(c, LBM_EINVAL, "d_f is NULL");
    if (!c->inited[comp]) return fail(c, LBM_ESTATE, "component has not been initialised");
    return c->vt->get_distributions(c, comp, d_f);
}

LBM_API int lbm_get_stream_map(lbm_ctx *c, int64_t *d_map) {
    CHECK_CTX(c);
    if (!d_map) return fail(c, LBM_EINVAL, "d_map is NULL");
    return c->vt->get_stream_map(c, d_map);
}

#define CUDA_TRY(c, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
    snprintf((c)->err, sizeof (c)->err, "%s: %s", #call, cudaGetErrorString(e_)); return LBM_ECUDA; } } while (0)

LBM_API int lbm_run_host(lbm_ctx *c, const uint8_t *h_mask, const void *const *h_rho0, const void *const *h_u0,
                         int n, void *h_rho_out, void *h_u_out) {
    CHECK_CTX(c);
    if (n < 0 || !h_rho0 || !h_u0) return fail(c, LBM_EINVAL, "bad arguments to lbm_run_host");
    for (int s = 0; s < c->ncomp; s++)
        if (!h_rho0[s] || !h_u0[s]) return fail(c, LBM_EINVAL, "h_rho0[s] / h_u0[s] is NULL");
    const size_t N = (size_t)c->g.N, rs = c->rs;
    uint8_t *d_mask = at<uint8_t>(c, c->lay.stage_mask);
    char *d_rho = c->ws + c->lay.stage_rho, *d_u = c->ws + c->lay.stage_u;
    // reset: new geometry allowed, nothing initialised
    c->geometry_frozen = false;
    c->inited[0] = c->inited[1] = false;
    c->cur = 0;
    if (h_mask) {
        CUDA_TRY(c, cudaMemcpyAsync(d_mask, h_mask, N, cudaMemcpyHostToDevice, c->stream));
    } else {
        CUDA_TRY(c, cudaMemsetAsync(d_mask, 0, N, c->stream));
    }
    if (int rc = lbm_set_geometry(c, d_mask)) return rc;
    for (int s = 0; s < c->ncomp; s++) {
        CUDA_TRY(c, cudaMemcpyAsync(d_rho, h_rho0[s], N * rs, cudaMemcpyHostToDevice, c->stream));
        CUDA_TRY(c, cudaMemcpyAsync(d_u, h_u0[s], c->D * N * rs, cudaMemcpyHostToDevice, c->stream));
        if (int rc = lbm_init_equilibrium(c, s, d_rho, d_u)) return rc;
    }
    if (int rc = lbm_step(c, n)) return rc;
    if (h_rho_out || h_u_out) {
        if (int rc = lbm_macro(c, 0, h_rho_out ? d_rho : nullptr, h_u_out ? d_u : nullptr)) return rc;
        if (h_rho_out) CUDA_TRY(c, cudaMemcpyAsync(h_rho_out, d_rho, N * rs, cudaMemcpyDeviceToHost, c->stream));
        if (h_u_out) CUDA_TRY(c, cudaMemcpyAsync(h_u_out, d_u, c->D * N * rs, cudaMemcpyDeviceToHost, c->stream));
    }
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return LBM_OK;
}

// ---- z-slab decomposition --------------------------------------------------------------
namespace {

template <typename T>
int copy_planes(lbm_ctx *to, cudaStream_t stream, const T *src, T *dst, int64_t Nsrc, int64_t Ndst, int from_plane, int to_plane,
                int ndir, const PlaneList &dirs) {
    const int plane = to->g.nx * to->g.ny;
    const dim3 grid((plane + 255) / 256, ndir);
    slab_copy_planes_kernel<T><<<grid, 256, 0, stream>>>(src, dst, Nsrc, Ndst, (int64_t)from_plane * plane, (int64_t)to_plane * plane,
                                                        plane, dirs);
    return check_launch(to, "slab_copy_planes_kernel");
}

// Fill the ghost plane `to_plane` of `to` from the interior plane `from_plane` of `from`, on `to`'s side stream.
// what = 0: the populations with e_z = ez of buffer `buf` (the one the step in progress writes) of every
// component; 1: the psi fields.
template <typename T> int fill_ghost(lbm_ctx *to, lbm_ctx *from, int from_plane, int to_plane, int ez, int what, int buf) {
    if (what == 1) {
        PlaneList one = {{0}};
        T *pa = at<T>(to, to->lay.psi[0]);
        const T *qa = at<T>(from, from->lay.psi[0]);
        for (int s = 0; s < 2; s++)  // planar psi_A | psi_B (split kernels)
            if (int rc = copy_planes<T>(to, to->slab_stream, qa + s * from->g.N, pa + s * to->g.N, from->g.N, to->g.N, from_plane, to_plane, 1, one))
                return rc;
        return LBM_OK;
    }
    PlaneList dirs = {{0}};
    int32_t e[3 * LBM_QMAX];
    int nd = 0;
    lbm_lattice_info(to->p.lattice, nullptr, nullptr, e, nullptr, nullptr);
    for (int i = 0; i < to->Q; i++)
        if (e[3 * i + 2] == ez) dirs.dir[nd++] = i;
    for (int s = 0; s < to->ncomp; s++)
        if (int rc = copy_planes<T>(to, to->slab_stream, at<T>(from, from->lay.store[s][buf]), at<T>(to, to->lay.store[s][buf]),
                                    from->g.N, to->g.N, from_plane, to_plane, nd, dirs)) return rc;
    return LBM_OK;
}

int fill_ghost_any(lbm_ctx *to, lbm_ctx *from, int from_plane, int to_plane, int ez, int what, int buf) {
    return to->rs == 4 ? fill_ghost<float>(to, from, from_plane, to_plane, ez, what, buf)
                       : fill_ghost<double>(to, from, from_plane, to_plane, ez, what, buf);
}

// Slabs may live on different devices: launches and event calls for a slab run with its device current.
struct DeviceGuard {
    int saved = -1;
    DeviceGuard() { if (cudaGetDevice(&saved) != cudaSuccess) saved = -1; }
    void use(const lbm_ctx *c) { if (c->device != current()) cudaSetDevice(c->device); }
    static int current() { int d = -1; cudaGetDevice(&d); return d; }
    ~DeviceGuard() { if (saved >= 0 && saved != current()) cudaSetDevice(saved); }
};

struct Slabs {
    lbm_ctx *const *c;
    int count, periodic;
    lbm_ctx *below(int k) const { return k > 0 ? c[k - 1] : (periodic ? c[count - 1] : nullptr); }
    lbm_ctx *above(int k) const { return k + 1 < count ? c[k + 1] : (periodic ? c[0] : nullptr); }
};

int slab_resources(lbm_ctx *c) {
    if (!c->slab_stream && cudaStreamCreateWithFlags(&c->slab_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(c, LBM_ECUDA, "cudaStreamCreate failed");
    if (!c->slab_event && cudaEventCreateWithFlags(&c->slab_event, cudaEventDisableTiming) != cudaSuccess) return fail(c, LBM_ECUDA, "cudaEventCreate failed");
    if (!c->slab_event2 && cudaEventCreateWithFlags(&c->slab_event2, cudaEventDisableTiming) != cudaSuccess) return fail(c, LBM_ECUDA, "cudaEventCreate failed");
    return LBM_OK;
}

// One pass (a whole step, or one phase of a Shan-Chen step) over every slab, the way section 3.6 of the
// paper orders it: the two boundary interior planes first; as soon as they are done, the ghost
// planes of the neighbours are filled from them on a side stream, concurrently with the bulk launch.
//   phase: sc_phase of the launches (0 whole step, 1 macro fields, 2 collide); what: 0 populations, 1 psi.
int slab_pass(const Slabs &S, DeviceGuard &dev, int phase, int what) {
    auto launch = [&](lbm_ctx *c, int z0, int zc) -> int {
        if (zc <= 0) return LBM_OK;
        c->zsel0 = z0; c->zselc = zc; c->no_advance = true; c->sc_phase = phase;
        const int rc = c->vt->step(c, 1);
        c->zsel0 = 0; c->zselc = c->g.nz; c->no_advance = false; c->sc_phase = 0;
        return rc;
    };
    for (int k = 0; k < S.count; k++) {  // boundary planes: local z = 1 and z = nz - 2
        lbm_ctx *c = S.c[k];
        dev.use(c);
        if (int rc = launch(c, 1, 1)) return rc;
        if (c->g.nz - 2 > 1) if (int rc = launch(c, c->g.nz - 2, 1)) return rc;
        if (cudaEventRecord(c->slab_event, c->stream) != cudaSuccess) return fail(c, LBM_ECUDA, "cudaEventRecord failed");
    }
    for (int k = 0; k < S.count; k++) {  // ghost planes <- the neighbours' fresh boundary planes (side stream)
        lbm_ctx *c = S.c[k], *below = S.below(k), *above = S.above(k);
        dev.use(c);
        const int buf = c->cur ^ 1;  // the buffer this step writes (ignored for psi)
        for (lbm_ctx *nb : {c, below, above})
            if (nb && cudaStreamWaitEvent(c->slab_stream, nb->slab_event, 0) != cudaSuccess) return fail(c, LBM_ECUDA, "cudaStreamWaitEvent failed");
        // lower ghost (plane 0) <- top interior plane of the slab below: what moves up (e_z = +1)
        if (below) if (int rc = fill_ghost_any(c, below, below->g.nz - 2, 0, +1, what, buf)) return rc;
        // upper ghost (plane nz-1) <- bottom interior plane (1) of the slab above: what moves down (e_z = -1)
        if (above) if (int rc = fill_ghost_any(c, above, 1, c->g.nz - 1, -1, what, buf)) return rc;
        if (cudaEventRecord(c->slab_event2, c->slab_stream) != cudaSuccess) return fail(c, LBM_ECUDA, "cudaEventRecord failed");
    }
    for (int k = 0; k < S.count; k++) {  // bulk planes 2 .. nz - 3, overlapping the copies
        lbm_ctx *c = S.c[k];
        dev.use(c);
        if (int rc = launch(c, 2, c->g.nz - 4)) return rc;
    }
    for (int k = 0; k < S.count; k++) {  // nobody goes on before its ghosts are filled and its planes have been read
        lbm_ctx *c = S.c[k];
        dev.use(c);
        for (lbm_ctx *nb : {c, S.below(k), S.above(k)})
            if (nb && cudaStreamWaitEvent(c->stream, nb->slab_event2, 0) != cudaSuccess) return fail(c, LBM_ECUDA, "cudaStreamWaitEvent failed");
    }
    return LBM_OK;
}

}  // namespace

LBM_API int lbm_step_slabs(lbm_ctx *const *slabs, int count, int periodic_z, int n) {
    if (!slabs || count < 1) return fail(nullptr, LBM_EINVAL, "slabs is NULL or count < 1");
    DeviceGuard dev;
    for (int k = 0; k < count; k++) {
        lbm_ctx *c = slabs[k];
        CHECK_CTX(c);
        if (n < 0) return fail(c, LBM_EINVAL, "n < 0");
        if (int rc = check_state(c)) return rc;
        if (c->p.lattice != LBM_D3Q19 || c->aa) return fail(c, LBM_EUNSUPPORTED, "slabs: D3Q19 with the AB store only");
        if (c->p.model == LBM_SC2 && !c->sc_split) return fail(c, LBM_EUNSUPPORTED, "slabs: Shan-Chen needs the split kernels");
        if (c->g.nz < 3) return fail(c, LBM_EINVAL, "slabs: a slab needs two ghost planes and at least one interior plane");
        const lbm_ctx *a = slabs[0];
        if (c->g.nx != a->g.nx || c->g.ny != a->g.ny || c->p.model != a->p.model || c->rs != a->rs || c->cur != a->cur || c->steps != a->steps)
            return fail(c, LBM_EINVAL, "slabs: contexts differ in nx, ny, model, precision or time step");
        dev.use(c);
        if (int rc = slab_resources(c)) return rc;
    }
    const Slabs S = {slabs, count, periodic_z};
    for (int t = 0; t < n; t++) {
        if (slabs[0]->p.model == LBM_SC2) {
            if (int rc = slab_pass(S, dev, 1, 1)) return rc;  // macro fields; psi planes exchanged (eq. 10 reads neighbours)
            if (int rc = slab_pass(S, dev, 2, 0)) return rc;  // collide; the crossing populations of the new state exchanged
        } else {
            if (int rc = slab_pass(S, dev, 0, 0)) return rc;
        }
        for (int k = 0; k < count; k++) { slabs[k]->cur ^= 1; slabs[k]->steps++; }
    }
    return LBM_OK;
}

LBM_API int lbm_get_counters(const lbm_ctx *c, int64_t *steps, int64_t *launches) {
    CHECK_CTX(c);
    if (steps) *steps = c->steps;
    if (launches) *launches = c->launches;
    return LBM_OK;
}

LBM_API int lbm_get_dispatch(const lbm_ctx *c, lbm_dispatch *out) {
    CHECK_CTX(c);
    if (!out) return LBM_EINVAL;
    out->nodes_per_thread = c->p.model == LBM_SC2 ? (c->sc_split ? c->sc_split : (c->vec >= 2 && c->rs == 4) ? 2 : 1) : c->vec;

    out->sc_split = c->p.model == LBM_SC2 && c->sc_split;
    out->index_bits = c->idx32 ? 32 : 64;
    out->graph_replay = (c->use_graph && !c->no_graph) ? GRAPH_STEPS : 0;
    out->resident_nodes_per_cta = (c->resident_slog2 > 0 && c->resident_state >= 0) ? 1 << c->resident_slog2 : 0;
    out->resident_ctas = out->resident_nodes_per_cta ? c->resident_ctas : 0;
    out->rows_per_block = (c->rows > 0 && !c->aa && c->p.model != LBM_SC2 && c->idx32 && c->vec <= 2) ? c->rows : 0;
    out->block_threads = c->block_threads;
    out->rows_strided = (out->rows_per_block > 0 && c->rows_strided && c->vec == 2) ? 1 : 0;
    return LBM_OK;
}

LBM_API const char *lbm_last_error(const lbm_ctx *c) { return c ? c->err : g_err; }
