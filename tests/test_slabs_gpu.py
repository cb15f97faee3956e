"""z-slab decomposition (NEXT-5; section 3.6 of the paper): one lattice split over several
contexts, each holding its planes plus one ghost plane on either side; lbm_step_slabs exchanges, after
every step, the 5 of 19 populations that cross each face (and the psi planes for Shan-Chen).  The
interior planes must hold exactly the bits of a single context that runs the whole lattice -- the
decomposition changes where a node is computed, not what is computed."""
import numpy as np
import pytest

from paper_1311_2404_b200 import workloads as W

pytestmark = pytest.mark.gpu


def slab_of(w, z0, nl):
    """Workload of global planes [z0, z0 + nl) with one ghost plane on each side (periodic seam)."""
    import copy
    idx = np.arange(z0 - 1, z0 + nl + 1) % w.nz
    s = copy.copy(w)
    s.nz = nl + 2
    s.mask = np.ascontiguousarray(w.mask[idx])
    s.rho = [np.ascontiguousarray(r[idx]) for r in w.rho]
    s.u = [np.ascontiguousarray(u[:, idx]) for u in w.u]
    return s


def run_split(B, w, cuts, steps, streams=None):
    import torch
    sims, z0 = [], 0
    for k, nl in enumerate(cuts):
        s = slab_of(w, z0, nl)
        sim = B.from_workload(s, stream=None if streams is None else streams[k])
        sim.set_geometry(s.mask)
        for c in range(w.ncomp):
            sim.init_equilibrium(s.rho[c], s.u[c], comp=c)
        sims.append(sim)
        z0 += nl
    assert z0 == w.nz
    torch.cuda.synchronize()
    for n in steps:
        B.lbm_step_slabs([s.ctx for s in sims], True, n)
    out = [torch.cat([s.get_distributions(c)[:, 1:-1] for s in sims], dim=1) for c in range(w.ncomp)]
    macro = [torch.cat([s.macro(c)[0][1:-1] for s in sims], dim=0) for c in range(w.ncomp)]
    torch.cuda.synchronize()
    for s in sims:
        s.close()
    return out, macro


def run_whole(B, w, steps):
    sim = B.from_workload(w)
    sim.set_geometry(w.mask)
    for c in range(w.ncomp):
        sim.init_equilibrium(w.rho[c], w.u[c], comp=c)
    for n in steps:
        for _ in range(n):
            sim.step(1)   # plain single launches: the slab path steps one launch at a time as well
    out = [sim.get_distributions(c).clone() for c in range(w.ncomp)]
    macro = [sim.macro(c)[0].clone() for c in range(w.ncomp)]
    sim.close()
    return out, macro


CASES = {
    "c2": lambda: W.c2_channel(64, 40, 36),
    "c3": lambda: W.c3_mrt_obstacles(48, 36, 30),
    "c5": lambda: W.c5_shan_chen(32, 24, 30),
    "c4": lambda: W.c4_duct(32, 20, 18),
}


@pytest.mark.parametrize("cfg,cuts", [("c2", (18, 18)), ("c2", (7, 20, 9)), ("c3", (11, 19)), ("c5", (15, 15)),
                                      ("c5", (1, 22, 7)), ("c4", (9, 9)), ("c2", (36,))])
def test_slab_split_is_bit_identical_to_the_single_context_run(B_, cfg, cuts):
    import torch
    B = B_
    w = CASES[cfg]()
    steps = [1, 2, 30]
    whole, mw = run_whole(B, w, steps)
    split, ms = run_split(B, w, cuts, steps)
    live = torch.from_numpy(w.mask != W.SOLID).to(whole[0].device)
    for c in range(w.ncomp):
        assert torch.equal(whole[c][:, live], split[c][:, live]), (cfg, cuts, c)
        assert torch.equal(mw[c], ms[c])


def test_slabs_on_different_streams(B_):
    import torch
    B = B_
    w = CASES["c5"]()
    whole, _ = run_whole(B, w, [25])
    streams = [torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()]
    split, _ = run_split(B, w, (10, 12, 8), [25], streams=streams)
    for c in range(2):
        assert torch.equal(whole[c], split[c])


def test_slab_errors(B_):
    B = B_
    w = CASES["c2"]()
    a = B.from_workload(slab_of(w, 0, 18))
    b = B.from_workload(slab_of(w, 18, 18))
    with pytest.raises(RuntimeError):          # not initialised
        B.lbm_step_slabs([a.ctx, b.ctx], True, 1)
    for s, z0 in ((a, 0), (b, 18)):
        sw = slab_of(w, z0, 18)
        s.set_geometry(sw.mask)
        s.init_equilibrium(sw.rho[0], sw.u[0])
    a.step(1)                                   # slabs out of step
    with pytest.raises(RuntimeError):
        B.lbm_step_slabs([a.ctx, b.ctx], True, 1)
    c1 = W.c1_taylor_green(32)
    d2 = B.from_workload(c1)
    d2.init_equilibrium(c1.rho[0], c1.u[0])
    with pytest.raises(RuntimeError):          # D2Q9 has no z
        B.lbm_step_slabs([d2.ctx], True, 1)
    for s in (a, b, d2):
        s.close()


@pytest.fixture(scope="module")
def B_():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1311_2404_b200 import binding
    binding.load()
    return binding
