"""Seeded randomised differential test: random lattice, model, precision, store, force scheme, extents
(including ragged and tiny ones), node types, relaxation rates and step counts, GPU (through the C ABI)
against the oracle.  It found the one bug the hand-written cases had missed (the Smagorinsky constant
was dropped when no body force was set)."""
import numpy as np
import pytest

from paper_1311_2404_b200 import workloads as W

pytestmark = pytest.mark.gpu


def random_case(rng):
    lat = int(rng.integers(0, 2))
    model = int(rng.choice([W.BGK, W.MRT, W.SC2, W.REG, W.LES]))
    prec, store, scheme = int(rng.integers(0, 2)), int(rng.integers(0, 2)), int(rng.integers(0, 2))
    nx, ny = int(rng.integers(1, 70)), int(rng.integers(1, 40))
    nz = 1 if lat == W.D2Q9 else int(rng.integers(1, 20))
    if rng.random() < 0.3:
        nx = int(rng.choice([4, 8, 16, 32, 64, 128]))       # extents that take the 2- and 4-node packs
    D = 2 if lat == W.D2Q9 else 3
    tau = (float(rng.uniform(0.55, 1.5)), float(rng.uniform(0.55, 1.5)))
    force = tuple(float(x) for x in rng.uniform(-2e-4, 2e-4, 3)) if rng.random() < 0.7 else (0.0, 0.0, 0.0)
    if D == 2:
        force = (force[0], force[1], 0.0)
    if model == W.REG and scheme == W.FORCE_GUO:
        force = (0.0, 0.0, 0.0)                              # reading A23
    ncomp = 2 if model == W.SC2 else 1
    seed = int(rng.integers(1_000_000))
    if rng.integers(0, 3) == 0:
        mask, rho, u = W.random_state(lat, nx, ny, nz, seed, solid_fraction=float(rng.choice([0, 0.05, 0.3])), ncomp=ncomp)
    else:
        mask, rho, u = W.random_types(lat, nx, ny, nz, seed, ncomp=ncomp)
    rates = None
    if model == W.MRT:
        rates = list(rng.uniform(0.8, 1.8, 9 if lat == W.D2Q9 else 19))
        for k in ((0, 3, 5) if lat == W.D2Q9 else (0, 3, 5, 7)):   # conserved moments: 0 or anything
            rates[k] = 0.0 if rng.random() < 0.5 else float(rng.uniform(0.8, 1.2))
    w = W.Workload("fuzz", lat, model, prec, nx, ny, nz, tau, 0, force=force, rates=rates,
                   sc_G=float(rng.uniform(-0.5, 0.9)), sc_psi=int(rng.integers(0, 2)),
                   bc_velocity=tuple(float(x) for x in rng.uniform(-0.03, 0.03, 3)) if D == 3 else (0.02, -0.01, 0.0),
                   force_scheme=scheme, smagorinsky_cs=float(rng.uniform(0, 0.2)))
    w.mask, w.rho, w.u = mask, rho, u
    return w, store, [int(rng.integers(1, 9)), int(rng.integers(1, 60))]


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_cases_against_oracle(orc, seed):
    import torch
    assert torch.cuda.is_available()
    from paper_1311_2404_b200 import binding as B
    rng = np.random.default_rng(seed)
    for case in range(60):
        w, store, chunks = random_case(rng)
        what = (seed, case, w.lattice, w.model, w.precision, store, w.force_scheme, (w.nx, w.ny, w.nz))
        sim = B.from_workload(w, store=store)
        ref = orc.Oracle(**w.params())
        sim.set_geometry(w.mask)
        ref.set_geometry(w.mask)
        for s in range(w.ncomp):
            sim.init_equilibrium(w.rho[s], w.u[s], comp=s)
            ref.init_equilibrium(w.rho[s], w.u[s], comp=s)
        assert np.array_equal(sim.get_stream_map().cpu().numpy(), ref.stream_map()), what
        assert np.array_equal(sim.get_geometry().cpu().numpy(), w.mask), what
        live = w.mask != W.SOLID
        for n in chunks:
            sim.step(n)
            ref.step(n)
            for s in range(w.ncomp):
                f_ref = ref.get_distributions(s)
                if np.abs(f_ref).max() > 10:       # a random parameter set the oracle itself cannot hold
                    break
                d = np.abs(sim.get_distributions(s).cpu().numpy().astype(np.float64) - f_ref)
                err = d[:, live].max() if live.any() else 0.0
                assert err <= (1e-5 if w.precision == W.F32 else 1e-12), (what, err)
        sim.close()


@pytest.mark.parametrize("seed", [21, 22])
def test_random_cases_with_random_forced_variants(orc, monkeypatch, seed):
    """The same random cases, each under a random draw of the test-only tuning knobs (pack width, row-walking
    kernel, split / monolithic Shan-Chen, graph replay, cluster-resident path, index width, block size), so
    that variant x model x store x geometry combinations no hand-written case lists still meet the oracle."""
    import torch
    assert torch.cuda.is_available()
    from paper_1311_2404_b200 import binding as B
    rng = np.random.default_rng(seed)
    monkeypatch.setenv("LBM_TUNING", "1")
    for case in range(120):
        w, store, chunks = random_case(rng)
        env = dict(LBM_VEC=str(rng.choice([1, 2, 4])), LBM_ROWS=str(rng.choice([0, 1, 2, 3])), LBM_SC_SPLIT=str(rng.integers(0, 2)),
                   LBM_NO_GRAPH=str(rng.integers(0, 2)), LBM_NO_RESIDENT=str(rng.integers(0, 2)), LBM_IDX64=str(int(rng.random() < 0.15)),
                   LBM_BLOCK_THREADS=str(rng.choice([32, 64, 128, 256])), LBM_SC_FIELDS_VEC=str(rng.integers(1, 3)),
                   LBM_ROWS_STRIDED=str(rng.integers(0, 2)))
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        what = (seed, case, w.lattice, w.model, w.precision, store, w.force_scheme, (w.nx, w.ny, w.nz), env)
        sim = B.from_workload(w, store=store)
        ref = orc.Oracle(**w.params())
        sim.set_geometry(w.mask)
        ref.set_geometry(w.mask)
        for s in range(w.ncomp):
            sim.init_equilibrium(w.rho[s], w.u[s], comp=s)
            ref.init_equilibrium(w.rho[s], w.u[s], comp=s)
        live = w.mask != W.SOLID
        for n in chunks + [int(rng.integers(50, 100))]:
            sim.step(n)
            ref.step(n)
            blown = False
            for s in range(w.ncomp):
                f_ref = ref.get_distributions(s)
                if not np.isfinite(f_ref).all() or np.abs(f_ref).max() > 10:       # the oracle itself cannot hold this draw
                    blown = True
                    break
                d = np.abs(sim.get_distributions(s).cpu().numpy().astype(np.float64) - f_ref)
                err = d[:, live].max() if live.any() else 0.0
                assert err <= (1e-5 if w.precision == W.F32 else 1e-12), (what, err)
            if blown:
                break
        sim.close()
