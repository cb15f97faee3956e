// lbm_steps.cuh -- host-side launch loops of the step kernels (rows a1-a12), included by the
// lbm_step_*.cu translation units, which instantiate one model each for one <lattice, real> pair.
#pragma once
#include "lbm_impl.cuh"

namespace {

template <class L, typename T> struct Steps {
    static const T *src(lbm_ctx *c, int s) { return at<T>(c, c->lay.store[s][c->cur]); }
    static T *dst(lbm_ctx *c, int s) { return at<T>(c, c->lay.store[s][c->cur ^ 1]); }
    static uint8_t *type(lbm_ctx *c) { return at<uint8_t>(c, c->lay.type); }
    static uint32_t *link(lbm_ctx *c) { return at<uint32_t>(c, c->lay.link); }
    // for the V-node step kernels: no type array to read when every node is BULK
    static const uint8_t *type_or_null(lbm_ctx *c) { return c->all_bulk ? nullptr : at<uint8_t>(c, c->lay.type); }

    template <int V, int MODEL, int FORCE> static int step_single_v(lbm_ctx *c, int n, const Relax<T> &rp) {
        // 64-bit slot indices (Q * N >= 2^32: more than 226 M D3Q19 nodes) are built for the AB kernels of
        // D3Q19 LBGK / MRT / split Shan-Chen only (lbm_create rejects other combinations at that size)
        if constexpr (L::Q == 19 && (MODEL == MODEL_BGK || MODEL == MODEL_MRT)) {
            if (!c->idx32) return step_single_vi<V, int64_t, MODEL, FORCE>(c, n, rp);
        }
        return step_single_vi<V, uint32_t, MODEL, FORCE>(c, n, rp);
    }

    template <int V, typename I, int MODEL, int FORCE> static int step_single_vi(lbm_ctx *c, int n, const Relax<T> &rp) {
        const Launch l = span_launch(c, V, c->aa ? AA_MAX_BLOCK : 256);
        if constexpr (sizeof(I) == 4) {
        if (c->aa) {  // in place: even steps are local, odd steps move data; V-node packs on both
            T *f = at<T>(c, c->lay.store[0][0]);
            bool strided = false;  // obstacle-rich geometry: odd steps with per-lane source select, nodes a warp apart
            if constexpr (V == 2) strided = c->rows > 0 && c->rows_strided;
            const int64_t half_row_threads = (int64_t)(c->g.nx / 2) * c->g.ny;
            const dim3 sgrid((unsigned)((half_row_threads + 63) / 64), 1, c->zselc);
            for (int t = 0; t < n; t++) {
                if (c->cur == 0) aa_even_kernel<L, T, V, I, MODEL, FORCE><<<l.grid, l.block, 0, c->stream>>>(c->g, type_or_null(c), f, rp);
                else if (strided) {
                    if constexpr (V == 2) aa_odd_strided_kernel<L, T, 2, I, MODEL, FORCE><<<sgrid, 64, 0, c->stream>>>(c->g, link(c), f, rp);
                }
                else aa_odd_kernel<L, T, V, I, MODEL, FORCE><<<l.grid, l.block, 0, c->stream>>>(c->g, type_or_null(c), link(c), f, rp);
                if (int rc = check_launch(c, "aa_step_kernel")) return rc;
                c->cur ^= 1;
                c->steps++;
            }
            return LBM_OK;
        }
        }
        if constexpr (V <= 2 && sizeof(I) == 4) {
            if constexpr (V == 2)
            if (c->rows > 0 && c->rows_strided) {  // ... with the thread's two nodes half a row apart
                const int bx = (c->span_bx > 0 && c->span_bx <= 128) ? c->span_bx : 64;
                const int64_t spans = (int64_t)(c->g.nx / 2) * ((c->g.ny + c->rows - 1) / c->rows);
                const dim3 grid((unsigned)((spans + bx - 1) / bx), 1, c->zselc);
                for (int t = 0; t < n; t++) {
                    step_rows_strided_kernel<L, T, 2, I, MODEL, FORCE><<<grid, bx, 0, c->stream>>>(launch_geom(c), link(c), src(c, 0), dst(c, 0), rp, c->rows);
                    if (int rc = check_launch(c, "step_rows_strided_kernel")) return rc;
                    if (c->no_advance) continue;
                    c->cur ^= 1;
                    c->steps++;
                }
                return LBM_OK;
            }
            if (c->rows > 0) {  // obstacle-rich geometry: row-walking kernel, link words one row ahead
                const int bx = (c->span_bx > 0 && c->span_bx <= 128) ? c->span_bx : 64;
                const int64_t spans = (int64_t)(c->g.nx / V) * ((c->g.ny + c->rows - 1) / c->rows);  // (x-pack, y-chunk) pairs per z-plane
                const dim3 grid((unsigned)((spans + bx - 1) / bx), 1, c->zselc);
                for (int t = 0; t < n; t++) {
                    step_rows_kernel<L, T, V, I, MODEL, FORCE><<<grid, bx, 0, c->stream>>>(launch_geom(c), link(c), src(c, 0), dst(c, 0), rp, c->rows);
                    if (int rc = check_launch(c, "step_rows_kernel")) return rc;
                    if (c->no_advance) continue;
                    c->cur ^= 1;
                    c->steps++;
                }
                return LBM_OK;
            }
        }
        for (int t = 0; t < n; t++) {
            step_kernel<L, T, V, I, MODEL, FORCE><<<l.grid, l.block, 0, c->stream>>>(launch_geom(c), type_or_null(c), link(c), src(c, 0), dst(c, 0), rp);
            if (int rc = check_launch(c, "step_kernel")) return rc;
            if (c->no_advance) continue;
            c->cur ^= 1;
            c->steps++;
        }
        return LBM_OK;
    }

    // Whole lbm_step(n) in one launch for lattices that fit the shared memory of one thread-block cluster.
    // The first call probes the launch (shared-memory opt-in, non-portable cluster size, at least one
    // co-schedulable cluster: a MIG/MPS slice may have too few SMs); if it cannot run, the context falls
    // back to the ordinary step kernels with graph replay for good.
    template <int MODEL, int FORCE, int THREADS, bool SFIX> static int launch_resident(lbm_ctx *c, int n, const Relax<T> &rp, bool *unavailable) {
        auto kernel = resident_kernel<L, T, MODEL, FORCE, THREADS, SFIX>;
        const size_t smem = 2 * (size_t)L::Q * ((size_t)1 << c->resident_slog2) * sizeof(T);
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = c->resident_ctas; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.gridDim = dim3(c->resident_ctas); cfg.blockDim = dim3(THREADS); cfg.dynamicSmemBytes = smem;
        cfg.stream = c->stream; cfg.attrs = attr; cfg.numAttrs = 1;
        if (c->resident_state == 0) {
            int clusters = 0;
            cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e == cudaSuccess && c->resident_ctas > 8) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (e == cudaSuccess) e = cudaOccupancyMaxActiveClusters(&clusters, kernel, &cfg);
            if (e != cudaSuccess || clusters < 1) {
                cudaGetLastError();
                c->resident_state = -1;
                *unavailable = true;
                return LBM_OK;
            }
            c->resident_state = 1;
        }
        const int after = c->cur ^ (n & 1);
        cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, c->g, c->resident_slog2, (const uint8_t *)type(c), (const uint32_t *)link(c),
                                           src(c, 0), at<T>(c, c->lay.store[0][after]), rp, n);
        if (e != cudaSuccess) return fail(c, LBM_ECUDA, "resident_kernel: %s", cudaGetErrorString(e));
        if (int rc = check_launch(c, "resident_kernel")) return rc;
        c->cur = after;
        c->steps += n;
        return LBM_OK;
    }

    template <int MODEL, int FORCE> static int step_resident(lbm_ctx *c, int n, const Relax<T> &rp, bool *unavailable) {
        if constexpr (L::Q == 9) {  // nodes per CTA == threads per CTA: the unrolled loop with immediate addresses
            if (c->resident_slog2 == 10) return launch_resident<MODEL, FORCE, 1024, true>(c, n, rp, unavailable);
        }
        if (c->resident_slog2 == 9) return launch_resident<MODEL, FORCE, 512, true>(c, n, rp, unavailable);
        return launch_resident<MODEL, FORCE, 512, false>(c, n, rp, unavailable);
    }

    template <int MODEL, int FORCE> static int step_single(lbm_ctx *c, int n, const Relax<T> &rp) {
        if (c->resident_slog2 > 0 && c->resident_state >= 0 && n >= 2 && !c->aa) {
            bool unavailable = false;
            const int rc = step_resident<MODEL, FORCE>(c, n, rp, &unavailable);
            if (!unavailable) return rc;
            c->resident_slog2 = 0;  // fall through to the step kernels, graphs from the next call on
            c->use_graph = c->g.N <= GRAPH_MAX_SITES;
        }
        if constexpr (sizeof(T) == 4 && MODEL == MODEL_BGK) {  // 4-node packs are built for LBGK only (pick_vec)
            if (c->vec == 4) return step_single_v<4, MODEL, FORCE>(c, n, rp);
        }
        if (c->vec == 2) return step_single_v<2, MODEL, FORCE>(c, n, rp);
        return step_single_v<1, MODEL, FORCE>(c, n, rp);
    }

    template <int V, int PSI> static int step_sc_v(lbm_ctx *c, int n) {
        if (c->p.force_scheme == LBM_FORCE_EDM)
            return step_sc_vf<V, uint32_t, PSI, FORCE_EDM>(c, n);
        return step_sc_vf<V, uint32_t, PSI, FORCE_GUO>(c, n);
    }

    // VF = nodes per thread of the macro-field pass, V = of the collide pass (chosen independently)
    template <int V, typename I, int PSI, int FS> static int step_sc_vf(lbm_ctx *c, int n) {
        if constexpr (sizeof(T) == 4) {
            if (c->sc_fields_vec == 2 && !c->aa) return step_sc_vi<2, V, I, PSI, FS>(c, n);
        }
        return step_sc_vi<1, V, I, PSI, FS>(c, n);
    }

    template <int VF, int V, typename I, int PSI, int FS> static int step_sc_vi(lbm_ctx *c, int n) {
        const Launch l = span_launch(c, V), lf = span_launch(c, VF);
        const Relax<T> rA = make_relax<T>(c, 0), rB = make_relax<T>(c, 1);
        auto *psi = at<typename Pair<T>::type>(c, c->lay.psi[0]);
        for (int t = 0; t < n; t++) {
            sc_fields_kernel<L, T, VF, I, PSI><<<lf.grid, lf.block, 0, c->stream>>>(c->g, type_or_null(c), link(c), src(c, 0), src(c, 1), psi);
            if (int rc = check_launch(c, "sc_fields_kernel")) return rc;
            sc_step_kernel<L, T, V, I, PSI, FS><<<l.grid, l.block, 0, c->stream>>>(
                c->g, type_or_null(c), link(c), src(c, 0), src(c, 1), dst(c, 0), dst(c, 1), psi, rA, rB, T(c->p.sc_G));
            if (int rc = check_launch(c, "sc_step_kernel")) return rc;
            c->cur ^= 1;
            c->steps++;
        }
        return LBM_OK;
    }

    // Split variant: one macro-field pass (psi_A, psi_B, u') + one collide pass per component.
    template <int V, typename I, int PSI, int FS> static int step_sc_split_vi(lbm_ctx *c, int n) {
        const Launch l = span_launch(c, V, c->aa ? AA_MAX_BLOCK : 256);
        const Relax<T> rA = make_relax<T>(c, 0), rB = make_relax<T>(c, 1);
        T *psiA = at<T>(c, c->lay.psi[0]), *psiB = psiA + c->g.N, *up = at<T>(c, c->lay.up);
        if constexpr (sizeof(I) == 4) {
        if (c->aa) {  // in place: `cur` is the parity
            T *fA = at<T>(c, c->lay.store[0][0]), *fB = at<T>(c, c->lay.store[1][0]);
            for (int t = 0; t < n; t++) {
                aa_sc_fields_split_kernel<L, T, V, I, PSI><<<l.grid, l.block, 0, c->stream>>>(
                    c->g, c->cur, type_or_null(c), link(c), fA, fB, psiA, psiB, up, rA.inv_tau, rB.inv_tau);
                if (int rc = check_launch(c, "aa_sc_fields_split_kernel")) return rc;
                aa_sc_collide_split_kernel<L, T, V, I, PSI, FS><<<l.grid, l.block, 0, c->stream>>>(
                    c->g, c->cur, type_or_null(c), link(c), fA, psiB, up, rA, T(c->p.sc_G));
                if (int rc = check_launch(c, "aa_sc_collide_split_kernel")) return rc;
                aa_sc_collide_split_kernel<L, T, V, I, PSI, FS><<<l.grid, l.block, 0, c->stream>>>(
                    c->g, c->cur, type_or_null(c), link(c), fB, psiA, up, rB, T(c->p.sc_G));
                if (int rc = check_launch(c, "aa_sc_collide_split_kernel")) return rc;
                c->cur ^= 1;
                c->steps++;
            }
            return LBM_OK;
        }
        }
        for (int t = 0; t < n; t++) {
            // sc_phase (lbm_step_slabs): 1 = macro-field pass only, 2 = collide passes only (the psi planes of the
            // slab's ghost layers are exchanged in between), 0 = the whole step
            if (c->sc_phase != 2) {
                sc_fields_split_kernel<L, T, V, I, PSI><<<l.grid, l.block, 0, c->stream>>>(
                    launch_geom(c), type_or_null(c), link(c), src(c, 0), src(c, 1), psiA, psiB, up, rA.inv_tau, rB.inv_tau);
                if (int rc = check_launch(c, "sc_fields_split_kernel")) return rc;
            }
            if (c->sc_phase == 1) continue;
            sc_collide_split_kernel<L, T, V, I, PSI, FS><<<l.grid, l.block, 0, c->stream>>>(
                launch_geom(c), type_or_null(c), link(c), src(c, 0), dst(c, 0), psiB, up, rA, T(c->p.sc_G));
            if (int rc = check_launch(c, "sc_collide_split_kernel")) return rc;
            sc_collide_split_kernel<L, T, V, I, PSI, FS><<<l.grid, l.block, 0, c->stream>>>(
                launch_geom(c), type_or_null(c), link(c), src(c, 1), dst(c, 1), psiA, up, rB, T(c->p.sc_G));
            if (int rc = check_launch(c, "sc_collide_split_kernel")) return rc;
            if (c->no_advance) continue;
            c->cur ^= 1;
            c->steps++;
        }
        return LBM_OK;
    }
    template <int V, int PSI> static int step_sc_split_v(lbm_ctx *c, int n) {
        if (c->p.force_scheme == LBM_FORCE_EDM)
        if constexpr (L::Q == 19) {
            if (!c->idx32)
                return c->p.force_scheme == LBM_FORCE_EDM ? step_sc_split_vi<V, int64_t, PSI, FORCE_EDM>(c, n)
                                                          : step_sc_split_vi<V, int64_t, PSI, FORCE_GUO>(c, n);
        }
        if (c->p.force_scheme == LBM_FORCE_EDM) return step_sc_split_vi<V, uint32_t, PSI, FORCE_EDM>(c, n);
        return step_sc_split_vi<V, uint32_t, PSI, FORCE_GUO>(c, n);
    }

    template <int PSI> static int step_sc(lbm_ctx *c, int n) {
        if (c->sc_split > 0 || c->aa) {  // the in-place store has the split variant only
            if constexpr (sizeof(T) == 4) {
                if (c->sc_split == 4) return step_sc_split_v<4, PSI>(c, n);
            }
            if (c->sc_split == 2 || (c->sc_split == 4 && sizeof(T) == 8)) return step_sc_split_v<2, PSI>(c, n);
            return step_sc_split_v<1, PSI>(c, n);
        }
        if constexpr (sizeof(T) == 4) {  // fp64 with two components and V = 2 would spill
            if (c->vec >= 2 && !c->aa) return step_sc_v<2, PSI>(c, n);
        }
        return step_sc_v<1, PSI>(c, n);
    }

    template <int MODEL> static int step_model(lbm_ctx *c, int n) {
        Relax<T> rp = make_relax<T>(c, 0);
        const bool force = c->p.force[0] != 0.0 || c->p.force[1] != 0.0 || c->p.force[2] != 0.0;
        const bool edm = c->p.force_scheme == LBM_FORCE_EDM;
        if (MODEL == MODEL_MRT)
            for (int k = 0; k < L::Q; k++) {  // M^-1 = M^T diag(1/|M_k|^2): rows are orthogonal (A5)
                rp.cr[k] = T(c->p.rates[k] / Mrt<L, T>::norm(k));
                rp.cs[k] = T((1.0 - 0.5 * c->p.rates[k]) / Mrt<L, T>::norm(k));
                rp.in[k] = T(1.0 / Mrt<L, T>::norm(k));
            }
        if (MODEL == MODEL_LES) rp.cs2x36 = T(36.0 * c->p.smagorinsky_cs * c->p.smagorinsky_cs);
        if (!force) return step_single<MODEL, FORCE_NONE>(c, n, rp);
        if (edm) return step_single<MODEL, FORCE_EDM>(c, n, rp);
        if constexpr (MODEL == MODEL_REG) return fail(c, LBM_EUNSUPPORTED, "regularized LBGK takes a body force through the EDM only");
        else return step_single<MODEL, FORCE_GUO>(c, n, rp);
    }

    static int step_shan_chen(lbm_ctx *c, int n) {
        return c->p.sc_psi == LBM_PSI_RHO ? step_sc<0>(c, n) : step_sc<1>(c, n);
    }
};

}  // namespace

// Which model a translation unit instantiates is chosen by the macro it defines before including
// this header: LBM_STEP_BGK, LBM_STEP_MRT, LBM_STEP_REG, LBM_STEP_LES or LBM_STEP_SC.
#if defined(LBM_STEP_BGK)
template <class L, typename T> int lbm_step_bgk(lbm_ctx *c, int n) { return Steps<L, T>::template step_model<MODEL_BGK>(c, n); }
#elif defined(LBM_STEP_MRT)
template <class L, typename T> int lbm_step_mrt(lbm_ctx *c, int n) { return Steps<L, T>::template step_model<MODEL_MRT>(c, n); }
#elif defined(LBM_STEP_REG)
template <class L, typename T> int lbm_step_reg(lbm_ctx *c, int n) { return Steps<L, T>::template step_model<MODEL_REG>(c, n); }
#elif defined(LBM_STEP_LES)
template <class L, typename T> int lbm_step_les(lbm_ctx *c, int n) { return Steps<L, T>::template step_model<MODEL_LES>(c, n); }
#elif defined(LBM_STEP_SC)
template <class L, typename T> int lbm_step_sc(lbm_ctx *c, int n) { return Steps<L, T>::step_shan_chen(c, n); }
#endif
