"""Every kernel variant the library can pick (pack width 1/2/4, 32- and 64-bit slot indices, the row-walking
kernel for obstacle-rich geometries on/off, graph replay on/off, cluster-resident path on/off) against the
oracle.  The variants are normally chosen from the lattice size and geometry; the test-only tuning
environment variables (include/lbm.h; honoured only with LBM_TUNING=1) force each one here so that none
ships untested, and lbm_get_dispatch confirms that the forced variant is the one that ran."""
import itertools

import numpy as np
import pytest

from paper_1311_2404_b200 import workloads as W

pytestmark = pytest.mark.gpu

# the Shan-Chen variant (split per-component collide kernels | one monolithic kernel) rides on the LBM_ROWS axis
ENVS = [dict(LBM_TUNING="1", LBM_VEC=v, LBM_IDX64=i, LBM_ROWS=r, LBM_NO_GRAPH=g, LBM_NO_RESIDENT=g,
             LBM_SC_SPLIT="1" if r == "0" else "0", LBM_SC_FIELDS_VEC="2" if g == "1" else "1",
             LBM_ROWS_STRIDED="1" if g == "0" else "0")
        for v, i, r, g in itertools.product(("1", "2", "4"), ("0", "1"), ("0", "3"), ("0", "1"))]


def cases():
    mask, rho, u = W.random_types(W.D3Q19, 64, 12, 9, seed=3)
    for model, precision, scheme in ((W.BGK, W.F32, W.FORCE_GUO), (W.MRT, W.F64, W.FORCE_EDM), (W.LES, W.F32, W.FORCE_GUO),
                                     (W.REG, W.F64, W.FORCE_EDM)):
        w = W.Workload("variants", W.D3Q19, model, precision, 64, 12, 9, (0.7, 0.7), 60, force=(1e-4, -2e-4, 1e-4),
                       rates=W.mrt_rates_d3q19(0.7) if model == W.MRT else None, bc_velocity=(0.02, 0.0, -0.01),
                       force_scheme=scheme, smagorinsky_cs=0.15)
        w.mask, w.rho, w.u = mask, rho, u
        yield w
    mask, rho, u = W.random_types(W.D3Q19, 32, 10, 6, seed=4, ncomp=2)
    w = W.Workload("variants_sc", W.D3Q19, W.SC2, W.F32, 32, 10, 6, (0.9, 1.1), 60, sc_G=0.7, force=(1e-5, 0, 0))
    w.mask, w.rho, w.u = mask, rho, u
    yield w


@pytest.mark.parametrize("env", ENVS, ids=lambda e: "v%s_i64%s_rows%s_nograph%s" % (e["LBM_VEC"], e["LBM_IDX64"], e["LBM_ROWS"], e["LBM_NO_GRAPH"]))
def test_forced_variant_matches_oracle(orc, monkeypatch, env):
    import torch
    assert torch.cuda.is_available()
    from paper_1311_2404_b200 import binding as B
    for k, v in env.items():
        monkeypatch.setenv(k, v)
    for w in cases():
        for store in (B.LBM_STORE_AB, B.LBM_STORE_AA):
            sim = B.from_workload(w, store=store)
            ref = orc.Oracle(**w.params())
            sim.set_geometry(w.mask)
            ref.set_geometry(w.mask)
            d = sim.dispatch()
            idx64 = env["LBM_IDX64"] == "1" and store == B.LBM_STORE_AB and w.model in (W.BGK, W.MRT, W.SC2)  # where built
            assert d["index_bits"] == (64 if idx64 else 32)
            assert (d["graph_replay"] == 0) == (env["LBM_NO_GRAPH"] == "1")
            if w.model == W.SC2:
                assert d["sc_split"] == (1 if env["LBM_SC_SPLIT"] == "1" or store == B.LBM_STORE_AA or idx64 else 0)
            if w.model != W.SC2:
                widest = 4 if (w.precision == W.F32 and w.model == W.BGK) else 2   # 4-node packs: fp32 LBGK only
                if int(env["LBM_VEC"]) <= (4 if w.precision == W.F32 else 2):   # a width the precision has no pack for is ignored
                    assert d["nodes_per_thread"] == min(int(env["LBM_VEC"]), widest)
                rows_ok = store == B.LBM_STORE_AB and not idx64 and d["nodes_per_thread"] <= 2
                assert d["rows_per_block"] == (int(env["LBM_ROWS"]) if rows_ok else 0)
                assert d["rows_strided"] == int(d["rows_per_block"] > 0 and d["nodes_per_thread"] == 2 and env["LBM_ROWS_STRIDED"] == "1")
            for s in range(w.ncomp):
                sim.init_equilibrium(w.rho[s], w.u[s], comp=s)
                ref.init_equilibrium(w.rho[s], w.u[s], comp=s)
            sim.step(61)
            ref.step(61)
            live = w.mask != W.SOLID
            for s in range(w.ncomp):
                d = np.abs(sim.get_distributions(s).cpu().numpy().astype(np.float64) - ref.get_distributions(s))
                assert d[:, live].max() <= (1e-5 if w.precision == W.F32 else 1e-12), (env, w.model, store)
            sim.close()
