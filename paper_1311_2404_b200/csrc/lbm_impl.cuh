// lbm_impl.cuh -- host-side context, workspace layout and the per-<lattice, real> kernel dispatch.
// Included by lbm_b200.cu (the C ABI) and by one small translation unit per <lattice, real> pair
// (lbm_impl_*.cu), so that the kernel instantiations compile in parallel.  Product code: shares
// nothing with oracle/.
#pragma once
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/lbm.h"
#include "lbm_kernels.cuh"

using namespace lbm;

namespace {

thread_local char g_err[256] = "";

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
    size_t store[2][2], type, link, counters, psi[2], up, stage_mask, stage_rho, stage_u, total;
};

struct Vtbl;

}  // namespace

struct lbm_ctx {
    lbm_params p;
    int Q, D, ncomp;
    size_t rs;  // sizeof(real)
    Geom g;
    cudaStream_t stream;
    int device;  // CUDA device current at lbm_create (the workspace and the stream belong to it)
    char *ws;
    Layout lay;
    int cur;  // which of the two buffers holds the current state (AB)
    bool inited[2];
    bool geometry_frozen;
    int64_t steps, launches;
    bool aa;            // LBM_STORE_AA: one buffer, `cur` is the step parity (0 even, 1 odd)
    int resident_slog2; // > 0: the AB store fits one cluster's shared memory; log2 of nodes per CTA
    int resident_ctas;  // CTAs of that cluster (8, or 16 = non-portable size)
    int resident_state; // 0 not probed yet, 1 launchable, -1 not launchable here (fall back for good)
    int span_bx;        // tuning: block width (threads along x) of the step kernels, 0 = default
    bool all_bulk;      // no node of the geometry is SOLID / BOUNDARY / special: the step kernels skip the type array
    // lbm_step_slabs only: the next vt->step call covers z-planes [zsel0, zsel0 + zselc) and, with no_advance,
    // neither flips the buffers nor counts a step (boundary planes are launched before the bulk)
    int zsel0, zselc;
    bool no_advance;
    cudaStream_t slab_stream;  // side stream of the ghost-plane copies, so that they overlap the bulk launch
    cudaEvent_t slab_event2;   // "this slab's ghost planes are filled"
    int sc_phase;       // lbm_step_slabs only: which part of a Shan-Chen step the next vt->step call runs (see lbm_steps.cuh)
    cudaEvent_t slab_event;  // lbm_step_slabs only: "this slab's kernels up to here are enqueued", created on first use
    int sc_split;       // Shan-Chen: > 0 = split variant (one collide launch per component), nodes per thread
    int sc_fields_vec;  // Shan-Chen: nodes per thread of the macro-field pass (the collide pass uses `vec`)
    int rows_strided;   // step_rows_strided_kernel instead of step_rows_kernel where nx allows (tuning: LBM_ROWS_STRIDED)
    int rows;           // > 0: obstacle-rich geometry (>= 20 % of the nodes not BULK): step_rows_kernel, rows per block
    bool idx32;         // Q * N < 2^32: slot numbers fit 32 bits (cheaper address arithmetic)
    int block_x;        // one-node-per-thread kernels: 1-D block along x
    int vec;            // nodes per thread of the step kernels (1, 2 or 4 consecutive x)
    int block_threads;  // threads per block of the step kernels
    const Vtbl *vt;
    // small lattices are launch-bound: GRAPH_STEPS steps are captured once per buffer
    // parity into a CUDA graph and replayed; capture happens on a private stream because the
    // caller's stream may be the legacy default stream, which cannot be captured.
    bool use_graph;
    bool no_graph;      // graph replay switched off (tuning knob, or no capture stream could be created)
    cudaStream_t capture_stream;
    cudaGraphExec_t graph[2];
    int64_t graph_launches;  // kernels inside one graph
    char err[256];
};

namespace {

struct Vtbl {
    int (*set_geometry)(lbm_ctx *, const uint8_t *);
    int (*init_equilibrium)(lbm_ctx *, int, const void *, const void *);
    int (*step)(lbm_ctx *, int);
    int (*macro)(lbm_ctx *, int, void *, void *);
    int (*get_distributions)(lbm_ctx *, int, void *);
    int (*set_distributions)(lbm_ctx *, int, const void *);
    int (*get_stream_map)(lbm_ctx *, int64_t *);
};

int fail(lbm_ctx *c, int code, const char *fmt, const char *detail = "") {
    char *dst = c ? c->err : g_err;
    snprintf(dst, 256, fmt, detail);
    return code;
}

constexpr int GRAPH_STEPS = 50;           // steps per captured graph (even: the buffer parity is restored)
constexpr int64_t GRAPH_MAX_SITES = 1 << 20;  // above this a step takes >> launch latency

void drop_graphs(lbm_ctx *c) {
    for (int k = 0; k < 2; k++)
        if (c->graph[k]) { cudaGraphExecDestroy(c->graph[k]); c->graph[k] = nullptr; }
}

int check_launch(lbm_ctx *c, const char *what) {
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(c->err, sizeof c->err, "%s: %s", what, cudaGetErrorString(e));
        return LBM_ECUDA;
    }
    return LBM_OK;
}

template <typename T> T *at(lbm_ctx *c, size_t off) { return reinterpret_cast<T *>(c->ws + off); }

dim3 grid_of(const lbm_ctx *c) { return dim3((c->g.nx + c->block_x - 1) / c->block_x, c->g.ny, c->g.nz); }

template <typename T> Relax<T> make_relax(const lbm_ctx *c, int comp) {
    Relax<T> r;
    set_bgk(r, c->p.tau[comp]);
    for (int a = 0; a < 3; a++) { r.g[a] = T(c->p.force[a]); r.ubc[a] = T(c->p.bc_velocity[a]); }
    for (int k = 0; k < 19; k++) r.cr[k] = r.cs[k] = r.in[k] = T(0);
    return r;
}

}  // namespace

// Entry points of the step kernels, one explicit instantiation per <lattice, real> in lbm_step_*.cu.
template <class L, typename T> int lbm_step_bgk(lbm_ctx *c, int n);
template <class L, typename T> int lbm_step_mrt(lbm_ctx *c, int n);
template <class L, typename T> int lbm_step_sc(lbm_ctx *c, int n);
template <class L, typename T> int lbm_step_reg(lbm_ctx *c, int n);
template <class L, typename T> int lbm_step_les(lbm_ctx *c, int n);

namespace {

// ---- per <lattice, real> implementation -------------------------------------------------------
struct Launch { dim3 grid, block; };

// Step kernels: V nodes per thread along x, 2-D blocks (bx packs) x (by rows).
Geom launch_geom(const lbm_ctx *c) { Geom g = c->g; g.z0 = c->zsel0; return g; }  // Geom of a (partial) step launch

// Step kernels: V nodes per thread along x; 1-D blocks over the packs of a z-plane (rows back to back).
Launch span_launch(const lbm_ctx *c, int V, int max_threads = 256) {
    const int64_t packs = (int64_t)(c->g.nx / V) * c->g.ny;
    int threads = c->block_threads < max_threads ? c->block_threads : max_threads;
    if (c->span_bx > 0 && c->span_bx <= max_threads) threads = c->span_bx;
    while (threads > 32 && threads / 2 >= packs) threads /= 2;
    Launch l;
    l.block = dim3(threads, 1, 1);
    l.grid = dim3((unsigned)((packs + threads - 1) / threads), 1, c->zselc);
    return l;
}

template <class L, typename T> struct Impl {
    static const T *src(lbm_ctx *c, int s) { return at<T>(c, c->lay.store[s][c->cur]); }
    static T *dst(lbm_ctx *c, int s) { return at<T>(c, c->lay.store[s][c->cur ^ 1]); }
    static uint8_t *type(lbm_ctx *c) { return at<uint8_t>(c, c->lay.type); }
    static uint32_t *link(lbm_ctx *c) { return at<uint32_t>(c, c->lay.link); }

    static int set_geometry(lbm_ctx *c, const uint8_t *d_mask) {
        unsigned *cnt = at<unsigned>(c, c->lay.counters);
        if (cudaMemsetAsync(cnt, 0, sizeof(unsigned), c->stream) != cudaSuccess) return fail(c, LBM_ECUDA, "cudaMemsetAsync(counters)");
        build_links_kernel<L><<<grid_of(c), c->block_x, 0, c->stream>>>(c->g, d_mask, type(c), link(c), cnt);
        drop_graphs(c);
        return check_launch(c, "build_links_kernel");
    }

    template <int MODE> static int aa_convert(lbm_ctx *c, int s, const void *in0, const void *in1, void *out0, void *out1) {
        const double hf = c->p.model == LBM_SC2 ? 0.0 : 0.5;  // SC2 reports the bare component velocity
        aa_convert_kernel<L, T, MODE><<<grid_of(c), c->block_x, 0, c->stream>>>(
            c->g, c->cur, type(c), link(c), at<T>(c, c->lay.store[s][0]), (const T *)in0, (const T *)in1, (T *)out0,
            (T *)out1, T(hf * c->p.force[0]), T(hf * c->p.force[1]), T(hf * c->p.force[2]));
        return check_launch(c, "aa_convert_kernel");
    }

    static int init_equilibrium(lbm_ctx *c, int s, const void *rho, const void *u) {
        if (c->aa) return aa_convert<2>(c, s, rho, u, nullptr, nullptr);
        init_equilibrium_kernel<L, T><<<grid_of(c), c->block_x, 0, c->stream>>>(
            c->g, type(c), link(c), (const T *)rho, (const T *)u, at<T>(c, c->lay.store[s][c->cur]));
        return check_launch(c, "init_equilibrium_kernel");
    }

    static int set_distributions(lbm_ctx *c, int s, const void *f) {
        if (c->aa) return aa_convert<0>(c, s, f, nullptr, nullptr, nullptr);
        set_distributions_kernel<L, T><<<grid_of(c), c->block_x, 0, c->stream>>>(
            c->g, type(c), link(c), (const T *)f, at<T>(c, c->lay.store[s][c->cur]));
        return check_launch(c, "set_distributions_kernel");
    }

    static int get_distributions(lbm_ctx *c, int s, void *f) {
        if (c->aa) return aa_convert<1>(c, s, nullptr, nullptr, f, nullptr);
        get_distributions_kernel<L, T><<<grid_of(c), c->block_x, 0, c->stream>>>(c->g, type(c), link(c), src(c, s), (T *)f);
        return check_launch(c, "get_distributions_kernel");
    }

    static int macro(lbm_ctx *c, int s, void *rho, void *u) {
        if (c->aa) return aa_convert<3>(c, s, nullptr, nullptr, rho, u);
        const bool sc = c->p.model == LBM_SC2;  // SC2: bare component velocity (lbm.h)
        macro_kernel<L, T><<<grid_of(c), c->block_x, 0, c->stream>>>(
            c->g, type(c), link(c), src(c, s), (T *)rho, (T *)u, sc ? T(0) : T(0.5 * c->p.force[0]),
            sc ? T(0) : T(0.5 * c->p.force[1]), sc ? T(0) : T(0.5 * c->p.force[2]));
        return check_launch(c, "macro_kernel");
    }

    static int get_stream_map(lbm_ctx *c, int64_t *map) {
        stream_map_kernel<L><<<grid_of(c), c->block_x, 0, c->stream>>>(c->g, type(c), link(c), map);
        return check_launch(c, "stream_map_kernel");
    }

    // The step kernels are instantiated in one translation unit per model (lbm_step_*.cu), so that
    // they compile in parallel; here only the dispatch.
    static int step(lbm_ctx *c, int n) {
        if (c->p.model == LBM_SC2) return lbm_step_sc<L, T>(c, n);
        if (c->p.model == LBM_BGK_REG) return lbm_step_reg<L, T>(c, n);
        if (c->p.model == LBM_BGK_LES) return lbm_step_les<L, T>(c, n);
        return c->p.model == LBM_MRT ? lbm_step_mrt<L, T>(c, n) : lbm_step_bgk<L, T>(c, n);
    }

    static const Vtbl *table() {
        static const Vtbl vt = {&Impl::set_geometry, &Impl::init_equilibrium, &Impl::step, &Impl::macro,
                                &Impl::get_distributions, &Impl::set_distributions, &Impl::get_stream_map};
        return &vt;
    }
};

}  // namespace

// One factory per translation unit lbm_impl_*.cu.
const void *lbm_impl_d2q9_f32();
const void *lbm_impl_d2q9_f64();
const void *lbm_impl_d3q19_f32();
const void *lbm_impl_d3q19_f64();
