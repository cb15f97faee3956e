"""Bit-exact integer work (node masks, streaming index maps), ABI state machine, host-buffer path,
and full-size checks in the launch configuration bench.py times."""
import numpy as np
import pytest

from paper_1311_2404_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_1311_2404_b200 import binding
    binding.load()
    return binding


@pytest.mark.parametrize("lattice,shape", [
    (W.D2Q9, (37, 23, 1)), (W.D2Q9, (128, 64, 1)), (W.D3Q19, (33, 17, 9)), (W.D3Q19, (64, 8, 5)),
    (W.D3Q19, (2, 2, 2)), (W.D3Q19, (1, 1, 1)), (W.D3Q19, (300, 3, 2))])
@pytest.mark.parametrize("solid", [0.0, 0.05, 0.4])
def test_mask_and_stream_map_bit_exact(B, orc, lattice, shape, solid):
    nx, ny, nz = shape
    mask, _, _ = W.random_state(lattice, nx, ny, nz, seed=100 + nx, solid_fraction=solid)
    sim = B.Lbm(lattice, W.BGK, W.F32, nx, ny, nz, tau=0.8)
    ref = orc.Oracle(lattice, W.BGK, nx, ny, nz, tau=0.8)
    sim.set_geometry(mask)
    ref.set_geometry(mask)
    assert np.array_equal(sim.get_geometry().cpu().numpy(), mask)
    m_gpu = sim.get_stream_map().cpu().numpy()
    m_ref = ref.stream_map()
    assert m_gpu.dtype == np.int64 and np.array_equal(m_gpu, m_ref)
    # permutation of FLUID slots (reading A8) => exact mass conservation
    live = m_gpu[m_gpu >= 0]
    assert len(np.unique(live)) == len(live)


def test_mask_values_round_trip_and_unknown_bytes_are_solid(B):
    sim = B.Lbm(W.D3Q19, W.BGK, W.F32, 8, 4, 2, tau=0.8)
    mask = np.zeros((2, 4, 8), np.uint8)
    mask[0, 1, 2], mask[1, 3, 7], mask[1, 0, 0], mask[0, 0, 5] = 255, 7, 2, 3
    sim.set_geometry(mask)
    want = mask.copy()
    want[mask > 3] = 1  # unknown values are SOLID; 2 = WALL_FULLWAY and 3 = VELOCITY come back as given
    assert np.array_equal(sim.get_geometry().cpu().numpy(), want)


def test_state_machine_errors(B):
    import torch
    sim = B.Lbm(W.D3Q19, W.SC2, W.F32, 8, 8, 8, tau=(1.0, 1.0), sc_G=0.5)
    with pytest.raises(B.LbmError) as e:
        sim.step(1)
    assert e.value.code == B.LBM_ESTATE
    rho, u = torch.ones(8, 8, 8), torch.zeros(3, 8, 8, 8)
    sim.init_equilibrium(rho, u, comp=0)
    with pytest.raises(B.LbmError) as e:  # component B still missing
        sim.step(1)
    assert e.value.code == B.LBM_ESTATE
    with pytest.raises(B.LbmError) as e:
        sim.set_geometry(np.zeros((8, 8, 8), np.uint8))
    assert e.value.code == B.LBM_ESTATE
    with pytest.raises(B.LbmError) as e:
        sim.init_equilibrium(rho, u, comp=2)
    assert e.value.code == B.LBM_EINVAL
    sim.init_equilibrium(rho, u, comp=1)
    sim.step(0)
    sim.step(2)
    steps, launches = sim.counters()
    assert steps == 2 and launches >= 4 + 2  # two kernels per Shan-Chen step
    with pytest.raises(B.LbmError) as e:
        sim.step(-1)
    assert e.value.code == B.LBM_EINVAL


def test_set_get_distributions_round_trip_bit_exact(B):
    """get(set(f)) == f on FLUID slots up to the f - w storage shift; 0 on SOLID (lbm.h)."""
    import torch
    mask, _, _ = W.random_state(W.D3Q19, 21, 13, 6, seed=5, solid_fraction=0.2)
    sim = B.Lbm(W.D3Q19, W.BGK, W.F64, 21, 13, 6, tau=0.8)
    sim.set_geometry(mask)
    g = torch.Generator().manual_seed(1)
    f = torch.rand((19, 6, 13, 21), generator=g, dtype=torch.float64)
    sim.set_distributions(f)
    back = sim.get_distributions().cpu()
    fluid = torch.from_numpy(mask == 0)
    assert (back[:, ~fluid] == 0).all()
    assert (back[:, fluid] - f[:, fluid]).abs().max() <= 2.3e-16


@pytest.mark.parametrize("cfg", ["c1", "c5"])
def test_graph_replay_is_bit_identical_to_single_launches(B, cfg):
    """Small lattices replay 50-step CUDA graphs (launch-bound regime): step(120) must give
    exactly the bits of 120 x step(1), which never reaches the graph threshold."""
    # 160^2 = 25600 nodes: above the cluster-resident limit (D2Q9: 16384), below the graph limit (2^20)
    w = W.c1_taylor_green(160) if cfg == "c1" else W.c5_shan_chen(24, 20, 16)
    out = []
    for chunks in ([120], [1] * 120, [50, 7, 63]):
        sim = B.from_workload(w)
        sim.set_geometry(w.mask)
        for s in range(w.ncomp):
            sim.init_equilibrium(w.rho[s], w.u[s], comp=s)
        assert sim.dispatch()["graph_replay"] == 50 and sim.dispatch()["resident_nodes_per_cta"] == 0
        for n in chunks:
            sim.step(n)
        assert sim.counters()[0] == 120
        out.append([sim.get_distributions(s).clone() for s in range(w.ncomp)])
        assert sim.counters()[1] >= 120 * w.ncomp
        sim.close()
    import torch
    for other in out[1:]:
        for a, b in zip(out[0], other):
            assert torch.equal(a, b)


def test_run_host_matches_device_calls_and_oracle(B, orc):
    import torch
    w = W.c2_channel(40, 24, 12)
    sim, ref = B.from_workload(w), orc.Oracle(**w.params())
    mask = torch.from_numpy(w.mask).pin_memory()
    rho0 = torch.from_numpy(w.rho[0]).float().pin_memory()
    u0 = torch.from_numpy(w.u[0]).float().pin_memory()
    rho, u = sim.run_host(mask, [rho0], [u0], 30)
    ref.set_geometry(w.mask)
    ref.init_equilibrium(w.rho[0], w.u[0])
    ref.step(30)
    rho_r, u_r = ref.macro()
    assert np.abs(rho.numpy() - rho_r).max() <= 1e-5 and np.abs(u.numpy() - u_r).max() <= 1e-5
    # a second call resets the state (lbm.h) and reproduces the first bit for bit
    rho2, u2 = sim.run_host(mask, [rho0], [u0], 30)
    assert torch.equal(rho, rho2) and torch.equal(u, u2)


# ---- full size, bench launch configuration ------------------------------------------------------------
def crop_periodic(a, centre, r):
    """(2r+1)^3 periodic crop of the last three axes around centre = (z, y, x)."""
    out = a
    for ax, c in zip((-3, -2, -1), centre):
        idx = np.arange(c - r, c + r + 1) % a.shape[ax]
        out = np.take(out, idx, axis=ax)
    return np.ascontiguousarray(out)


@pytest.mark.parametrize("cfg,n", [("c2", 5), ("c3", 4), ("c4", 4), ("c5", 4), ("ldc", 5)])
def test_full_size_sampled_against_oracle(B, orc, cfg, n):
    """Full BASELINE.json size, as bench.py launches it.  Information moves one node per step, so
    f(x, n) depends only on the (2n+1)^3 box around x: the oracle recomputes sampled nodes one by
    one on periodic crops of the same seeded inputs (radius n+1; 2n+1 for Shan-Chen).  Plus mass conservation."""
    w = W.CONFIGS[cfg]()
    sim = B.from_workload(w)
    sim.set_geometry(w.mask)
    for s in range(w.ncomp):
        sim.init_equilibrium(w.rho[s], w.u[s], comp=s)
    fluid = w.mask != W.SOLID  # every node that holds populations
    m0 = [float(sim.macro(s)[0].double().sum()) for s in range(w.ncomp)]
    sim.step(n)
    rng = np.random.Generator(np.random.PCG64(7))
    pts = [(0, 1, 0), (w.nz - 1, w.ny - 2, w.nx - 1), (w.nz // 2, 1, w.nx // 2), (w.nz // 2, w.ny - 3, 2)]
    pts += [tuple(int(rng.integers(0, d)) for d in (w.nz, w.ny, w.nx)) for _ in range(9)]
    pts = [p for p in pts if fluid[p]]
    r = (2 * n if w.model == W.SC2 else n) + 1  # Shan-Chen reads neighbour densities: 2 nodes/step
    f_gpu = [sim.get_distributions(s) for s in range(w.ncomp)]
    tol = 1e-6 if w.precision == W.F32 else 1e-13
    for p in pts:
        kw = w.params()
        kw.update(nx=2 * r + 1, ny=2 * r + 1, nz=2 * r + 1)
        ref = orc.Oracle(**kw)
        ref.set_geometry(crop_periodic(w.mask, p, r))
        for s in range(w.ncomp):
            ref.init_equilibrium(crop_periodic(w.rho[s], p, r), crop_periodic(w.u[s], p, r), comp=s)
        ref.step(n)
        for s in range(w.ncomp):
            got = f_gpu[s][:, p[0], p[1], p[2]].double().cpu().numpy()
            want = ref.get_distributions(s)[:, r, r, r]
            assert np.abs(got - want).max() <= tol, (cfg, p, s)
    del f_gpu
    if cfg == "ldc":
        return  # the equilibrium-velocity lid exchanges mass with the flow by construction
    for s in range(w.ncomp):  # mass of each component is conserved (A8 permutation; A13)
        m1 = float(sim.macro(s)[0].double().sum())
        assert abs(m1 - m0[s]) <= (2e-7 if w.precision == W.F32 else 1e-13) * m0[s]


@pytest.mark.parametrize("lattice,shape,model,ctas", [
    (W.D2Q9, (64, 64, 1), W.BGK, 8), (W.D2Q9, (50, 37, 1), W.MRT, 8), (W.D3Q19, (16, 16, 16), W.BGK, 8),
    (W.D3Q19, (13, 9, 7), W.LES, 8), (W.D2Q9, (128, 128, 1), W.BGK, 16), (W.D2Q9, (96, 70, 1), W.MRT, 16),
    (W.D2Q9, (101, 150, 1), W.REG, 16)])
def test_cluster_resident_path_matches_single_launches_and_oracle(B, orc, lattice, shape, model, ctas):
    """Lattices of up to 4096 nodes (D2Q9: 16384, in a 16-CTA cluster) run lbm_step(n) as ONE launch of a
    thread-block cluster that keeps both buffers in distributed shared memory: must equal n single-step
    launches bit for bit (same arithmetic, same streaming rule) and the oracle within tolerance; all
    node types included."""
    import torch
    nx, ny, nz = shape
    mask, rho, u = W.random_types(lattice, nx, ny, nz, seed=91)
    D = 2 if lattice == W.D2Q9 else 3
    rates = (W.mrt_rates_d3q19(0.7) if lattice == W.D3Q19 else W.mrt_rates_d2q9(0.7)) if model == W.MRT else None
    w = W.Workload("resident", lattice, model, W.F64, nx, ny, nz, (0.7, 0.7), 60, rates=rates, smagorinsky_cs=0.15,
                   force=(1e-5, -2e-5, 3e-5 if D == 3 else 0.0), bc_velocity=(0.02, -0.01, 0.0),
                   force_scheme=W.FORCE_EDM if model == W.REG else W.FORCE_GUO)
    w.mask, w.rho, w.u = mask, rho, u
    out = []
    for chunks in ([60], [1] * 60, [7, 53]):
        sim = B.from_workload(w)
        sim.set_geometry(w.mask)
        sim.init_equilibrium(w.rho[0], w.u[0])
        assert sim.dispatch()["resident_ctas"] == ctas and sim.dispatch()["graph_replay"] == 0
        l0 = sim.counters()[1]
        for n in chunks:
            sim.step(n)
        assert sim.counters()[0] == 60
        if chunks == [60]:
            assert sim.counters()[1] - l0 == 1      # one kernel for all 60 steps
        out.append(sim.get_distributions().clone())
        sim.close()
    assert torch.equal(out[0], out[1]) and torch.equal(out[0], out[2])
    ref = orc.Oracle(**w.params())
    ref.set_geometry(w.mask)
    ref.init_equilibrium(w.rho[0], w.u[0])
    ref.step(60)
    live = w.mask != W.SOLID
    assert np.abs(out[0].cpu().numpy() - ref.get_distributions())[:, live].max() <= 1e-12


def test_runs_on_a_caller_stream(B, orc):
    """All work goes to the cudaStream_t given to lbm_create (lbm.h): a non-default torch stream,
    including the cluster-resident path (96^2 D2Q9), the graph-replay path (160^2) and a full-kernel path
    (40 x 24 x 12 D3Q19)."""
    import torch
    side = torch.cuda.Stream()
    for w in (W.c1_taylor_green(96), W.c1_taylor_green(160), W.c2_channel(40, 24, 12)):
        ref = orc.Oracle(**w.params())
        ref.set_geometry(w.mask)
        ref.init_equilibrium(w.rho[0], w.u[0])
        ref.step(120)
        with torch.cuda.stream(side):
            sim = B.from_workload(w, stream=side)
            sim.set_geometry(w.mask)
            sim.init_equilibrium(w.rho[0], w.u[0])
            sim.step(120)
            f = sim.get_distributions()
        side.synchronize()
        fluid = w.mask == 0
        assert np.abs(f.cpu().numpy().astype(np.float64) - ref.get_distributions())[:, fluid].max() <= 1e-5
        sim.close()
